// kcs_projector.cu -- layout transposes, ray-driven forward projector (+ fused Poisson ratio), exact-transpose
// gather back-projector (+ fused OSL update), sensitivity images.  sm_100a.
//
// Cited passages: P:<n> = PAPER.md line n; readings P1-P5, O1-O2, Q* are listed in DESIGN.md section 3.
//
// Design: activity and sinograms are kept frame-innermost, so the Tp frames of one pixel
// are one contiguous 16*Tp/4-byte run (one 128 B line at Tp = 32).  FG = Tp/FPT neighbouring lanes share one
// ray sample (forward) or one voxel (backward); each lane owns FPT frames as float4 registers.  Geometry math is
// frame-independent and amortised over the FPT frames; coalescing comes from the frame axis and therefore does
// not depend on the projection angle.
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

// ---------------------------------------------------------------------------------------------------------
// pack / unpack: planar [nf][rows][W]  <->  inner [dst_index][Tp]
// ---------------------------------------------------------------------------------------------------------
struct PackMap {
    long long nrows;
    int W;
    int rps;         // rows per slab
    long long slab;  // dst pixels per slab
    int rstride;     // dst pixels per row
    int off;         // dst pixel offset of (row 0, col 0) inside a slab
};

// rows and slabs fit 32 bits (kcs_launch_pack checks); Tp is a power of two (round_up4), lt = log2(Tp)
__device__ __forceinline__ size_t pack_dst(const PackMap &m, unsigned row, int col) {
    const unsigned s = row / (unsigned)m.rps, rr = row - s * (unsigned)m.rps;
    return (size_t)s * (size_t)m.slab + (size_t)rr * m.rstride + m.off + col;
}

// block (32, 8): one row segment of 32 columns, all frames.
__global__ void __launch_bounds__(256) k_pack(const float *__restrict__ src, size_t fs, int nf, float *__restrict__ dst, int Tp, int lt,
                                              PackMap m) {
    __shared__ float tile[KCS_MAX_FRAMES][33];
    const int c0 = blockIdx.x * 32;
    const unsigned row = blockIdx.y + blockIdx.z * gridDim.y;
    if (row >= (unsigned)m.nrows) return;
    const int tx = threadIdx.x, ty = threadIdx.y;
    const float *sp = src + (size_t)row * m.W + c0 + tx;
    for (int f = ty; f < Tp; f += 8) tile[f][tx] = (f < nf && c0 + tx < m.W) ? sp[(size_t)f * fs] : 0.f;
    __syncthreads();
    const int ncol = min(32, m.W - c0);
    float *dp = dst + pack_dst(m, row, c0) * Tp;
    const int n = ncol << lt;
    for (int e = ty * 32 + tx; e < n; e += 256) dp[e] = tile[e & (Tp - 1)][e >> lt];
}

__global__ void __launch_bounds__(256) k_unpack(const float *__restrict__ src, int Tp, int lt, float *__restrict__ dst, size_t fs, int nf,
                                                PackMap m) {
    __shared__ float tile[KCS_MAX_FRAMES][33];
    const int c0 = blockIdx.x * 32;
    const unsigned row = blockIdx.y + blockIdx.z * gridDim.y;
    if (row >= (unsigned)m.nrows) return;
    const int tx = threadIdx.x, ty = threadIdx.y;
    const int ncol = min(32, m.W - c0);
    const float *sp = src + pack_dst(m, row, c0) * Tp;
    const int n = ncol << lt;
    for (int e = ty * 32 + tx; e < n; e += 256) tile[e & (Tp - 1)][e >> lt] = sp[e];
    __syncthreads();
    float *dp = dst + (size_t)row * m.W + c0 + tx;
    if (c0 + tx < m.W)
        for (int f = ty; f < nf; f += 8) dp[(size_t)f * fs] = tile[f][tx];
}

static void pack_grid(long long nrows, int W, dim3 &grid) {
    const long long gy = nrows < 32768 ? nrows : 32768;
    grid = dim3((unsigned)((W + 31) / 32), (unsigned)gy, (unsigned)((nrows + gy - 1) / gy));
}

int kcs_launch_pack(kcs_ctx *c, const float *src, size_t fs, int nf, float *dst, int Tp, long long nrows, int W,
                    int rps, long long slab, int rstride, int off) {
    if (nrows >= (1LL << 31)) { c->err = "kcs_launch_pack: more than 2^31 rows"; return KCS_ERR_SHAPE; }
    PackMap m{nrows, W, rps, slab, rstride, off};
    dim3 grid;
    pack_grid(nrows, W, grid);
    ProfScope ps(c, KCS_K_PACK);
    int lt = 2;
    while ((1 << lt) < Tp) ++lt;
    k_pack<<<grid, dim3(32, 8), 0, c->stream>>>(src, fs, nf, dst, Tp, lt, m);
    LAUNCH_CHECK(c);
    return KCS_OK;
}

int kcs_launch_unpack(kcs_ctx *c, const float *src, int Tp, float *dst, size_t fs, int nf, long long nrows, int W,
                      int rps, long long slab, int rstride, int off) {
    if (nrows >= (1LL << 31)) { c->err = "kcs_launch_unpack: more than 2^31 rows"; return KCS_ERR_SHAPE; }
    PackMap m{nrows, W, rps, slab, rstride, off};
    dim3 grid;
    pack_grid(nrows, W, grid);
    ProfScope ps(c, KCS_K_UNPACK);
    int lt = 2;
    while ((1 << lt) < Tp) ++lt;
    k_unpack<<<grid, dim3(32, 8), 0, c->stream>>>(src, Tp, lt, dst, fs, nf, m);
    LAUNCH_CHECK(c);
    return KCS_OK;
}

// ---------------------------------------------------------------------------------------------------------
// Forward projector  (P1-P3; P:64-67 denominator of eq. 2; O1 for the fused ratio)
// ---------------------------------------------------------------------------------------------------------
struct FwdArgs {
    const float *xi;
    float *qi;
    const float *yi;     // packed measured sinogram [nz][A][B][Tp]       (ratio only)
    const float *ri;     // packed randoms, same layout                    (ratio, KCS_R_FULL)
    const float *r_pad;  // [32] per-frame randoms, 0 beyond T             (ratio, KCS_R_PER_FRAME)
    const float *mult;   // [nz][A][B] multiplicative sinogram (attenuation x normalisation) or NULL  (ratio only)
    int Tp, FG, BINS, KSPLIT, KCH, FB;
    int As, subset;
    int ratio, r_mode;
    float scale;
    float clip_r2;       // >= 0: x is zero outside a centred circle of this squared radius (mm^2)
};

#define KCS_ANCHOR 16  // steps between fp64 re-anchoring of the sample coordinates
#define KCS_FWD_UNROLL 2  // x 6 CTAs per SM: 3.02 ms per C4 subset launch; 1..8 x 1..8 CTAs all land within 4 % (3.02-3.13), 8 x 1: 3.62
#define KCS_FWD_TPB 128
#define KCS_BACK_TPB 128  // 4 CTAs of 128 threads per SM (128 registers): 2.64 ms per C4 subset launch against 2.71 with 2 x 256

// One thread = one ray x 4 frames; the FG = Tp/4 lanes of a ray read a whole pixel (16 FG bytes) per tap in one request.
template <int FG>
__global__ void __launch_bounds__(KCS_FWD_TPB, 6) k_forward(KGeom g, FwdArgs p) {
    constexpr int FPT = 4, Tp = 4 * FG;
    // 8 loads in flight per thread when a warp covers few rays (FG >= 4); with 16-32 rays per warp the extra
    // registers cost more occupancy than the unrolling hides (C5(a) at 1 and 4 frames per launch)
    constexpr int kUnroll = FG >= 4 ? KCS_FWD_UNROLL : 1;
    extern __shared__ float red[];
    const int tid = threadIdx.x;
    const int fg = tid % FG;
    const int bl = (tid / FG) % p.BINS;
    const int kc = tid / (FG * p.BINS);
    const int b = blockIdx.x * p.BINS + bl;
    const int la = blockIdx.y, z = blockIdx.z;
    const int a = p.subset < 0 ? la : p.subset + la * g.S;

    float acc[FPT];
#pragma unroll
    for (int f = 0; f < FPT; ++f) acc[f] = 0.f;

    if (b < g.B) {
        const double4 fw = g.fwd[a];
        const double bc = (double)b - g.cb;
        // Sample coordinates advance along the ray as 32-bit fixed point with FB fractional bits (2^-22 pixel at
        // image sizes <= 480), re-anchored from fp64 every KCS_ANCHOR steps: floor = shift, fraction = mask, and the
        // fraction becomes a float by placing it in the mantissa of [1,2) -- no conversions, no floorf.  The bilinear
        // interpolant is continuous (P2), so the <= 2e-6 pixel drift inside a block only perturbs the value by O(eps).
        const int FB = p.FB, msh = 23 - FB;
        const double qs = (double)(1 << FB);
        const int dxq = __double2int_rn(fw.y * qs), dyq = __double2int_rn(fw.w * qs);
        const unsigned fmask = (1u << FB) - 1u;
        // Ray clipping: padded coordinates P = index + KCS_PAD.  A sample contributes iff floor(P) in [PAD-1, PAD+n-1];
        // the loop runs over the k with P in [PAD - 1.5, PAD + n + 0.5) in both axes (a half-pixel margin that dwarfs the
        // fixed-point drift): every tap of such a sample lies inside the padded slice and the extra samples read zeros.
        const double pxa = fma(-g.ck, fw.y, fma(bc, fw.x, g.cx + (double)KCS_PAD));  // P_x at k = 0
        const double pya = fma(-g.ck, fw.w, fma(bc, fw.z, g.cy + (double)KCS_PAD));
        double tlo = (double)(kc * p.KCH), thi = (double)(min(g.K, (kc + 1) * p.KCH) - 1);
        {
            const double lo = (double)KCS_PAD - 1.5, hx = (double)(KCS_PAD + g.nx) + 0.5, hy = (double)(KCS_PAD + g.ny) + 0.5;
            if (fabs(fw.y) < 1e-9) { if (!(pxa >= lo && pxa < hx)) thi = -1.0; }
            else { const double t0 = (lo - pxa) / fw.y, t1 = (hx - pxa) / fw.y; tlo = fmax(tlo, fmin(t0, t1) + 1e-6); thi = fmin(thi, fmax(t0, t1) - 1e-6); }
            if (fabs(fw.w) < 1e-9) { if (!(pya >= lo && pya < hy)) thi = -1.0; }
            else { const double t0 = (lo - pya) / fw.w, t1 = (hy - pya) / fw.w; tlo = fmax(tlo, fmin(t0, t1) + 1e-6); thi = fmin(thi, fmax(t0, t1) - 1e-6); }
        }
        if (p.clip_r2 >= 0.f) {  // samples farther than the mask radius + 1.5 voxels from the axis only see zeros
            const double sb = bc * (double)g.bin_mm, h2 = (double)p.clip_r2 - sb * sb;
            if (h2 < 0.0) thi = -1.0;
            else { const double h = sqrt(h2) / (double)g.step_mm; tlo = fmax(tlo, g.ck - h); thi = fmin(thi, g.ck + h); }
        }
        const int k_lo = (int)ceil(tlo);       // clip bounds were moved 1e-6 steps inwards: strictly inside the margin
        const int k_hi = (int)floor(thi) + 1;
        const int rowstride = g.nxp * Tp;
        // taps are addressed as (CTA-uniform slice base) + (32-bit byte offset): one IMAD pair per sample instead of 64-bit
        // pointer arithmetic per tap (a padded slice is < 4 GB)
        const char *slice = reinterpret_cast<const char *>(p.xi + (size_t)z * g.nyp * rowstride);
        const unsigned rsb = (unsigned)rowstride * 4u, psb = (unsigned)Tp * 4u, fgb = (unsigned)fg * (FPT * 4u);
        // Anchor blocks sit on the absolute grid k = 0, 16, 32, ...: the fixed-point coordinates of sample k do not depend
        // on where clipping (or the K-split) starts the walk, so a clipped and an unclipped projection of an image that is
        // zero outside the field of view agree bit for bit.
        for (int kb = (k_lo / KCS_ANCHOR) * KCS_ANCHOR; kb < k_hi; kb += KCS_ANCHOR) {
            // fp64 anchor (P2): padded continuous index of sample (b, kb), advanced exactly to the first sample of the walk
            const double kk = (double)kb;
            const int k0 = max(kb, k_lo);
            int fxq = __double2int_rn(fma(kk, fw.y, pxa) * qs) + (k0 - kb) * dxq;
            int fyq = __double2int_rn(fma(kk, fw.w, pya) * qs) + (k0 - kb) * dyq;
            const int mmax = min(kb + KCS_ANCHOR, k_hi) - k0;
#pragma unroll(kUnroll)
            for (int m = 0; m < mmax; ++m) {
                const int i0 = fxq >> FB, j0 = fyq >> FB;
                const float wx = __uint_as_float((((unsigned)fxq & fmask) << msh) | 0x3f800000u) - 1.f;
                const float wy = __uint_as_float((((unsigned)fyq & fmask) << msh) | 0x3f800000u) - 1.f;
                const unsigned bo = (unsigned)j0 * rsb + (unsigned)i0 * psb + fgb, bo1 = bo + rsb;
                const float w11 = wx * wy, w10 = wx - w11, w01 = wy - w11, w00 = (1.f - wx) - w01;
                const float4 v00 = __ldg(reinterpret_cast<const float4 *>(slice + bo)),
                             v10 = __ldg(reinterpret_cast<const float4 *>(slice + bo + psb)),
                             v01 = __ldg(reinterpret_cast<const float4 *>(slice + bo1)),
                             v11 = __ldg(reinterpret_cast<const float4 *>(slice + bo1 + psb));
                acc[0] = fmaf(w11, v11.x, fmaf(w01, v01.x, fmaf(w10, v10.x, fmaf(w00, v00.x, acc[0]))));
                acc[1] = fmaf(w11, v11.y, fmaf(w01, v01.y, fmaf(w10, v10.y, fmaf(w00, v00.y, acc[1]))));
                acc[2] = fmaf(w11, v11.z, fmaf(w01, v01.z, fmaf(w10, v10.z, fmaf(w00, v00.z, acc[2]))));
                acc[3] = fmaf(w11, v11.w, fmaf(w01, v01.w, fmaf(w10, v10.w, fmaf(w00, v00.w, acc[3]))));
                fxq += dxq;
                fyq += dyq;
            }
        }
    }

    // combine the KSPLIT partial sums of a ray (fixed order: deterministic)
    if (p.KSPLIT > 1) {
        const int nbf = p.BINS * FG;
        const int idx = bl * FG + fg;
        if (kc > 0) {
#pragma unroll
            for (int f = 0; f < FPT; ++f) red[((kc - 1) * FPT + f) * nbf + idx] = acc[f];
        }
        __syncthreads();
        if (kc == 0) {
            for (int s = 1; s < p.KSPLIT; ++s)
#pragma unroll
                for (int f = 0; f < FPT; ++f) acc[f] += red[((s - 1) * FPT + f) * nbf + idx];
        }
    }
    if (kc != 0 || b >= g.B) return;

    const size_t o = (((size_t)z * p.As + la) * g.B + b) * Tp + fg * FPT;
    if (!p.ratio) {
#pragma unroll
        for (int q = 0; q < FPT / 4; ++q)
            reinterpret_cast<float4 *>(p.qi + o)[q] = make_float4(g.step_mm * acc[4 * q], g.step_mm * acc[4 * q + 1],
                                                                  g.step_mm * acc[4 * q + 2], g.step_mm * acc[4 * q + 3]);
    } else {
        // O1: yhat = scale A_s x + r ; q = y / yhat where yhat > 1e-12 else 0
        const size_t oy = (((size_t)z * g.A + a) * g.B + b) * Tp + fg * FPT;
        // S8(f)3: yhat = scale n (A x) + r and the transpose acts on n q (n = attenuation x normalisation of this ray)
        const float nm = p.mult ? __ldg(p.mult + ((size_t)z * g.A + a) * g.B + b) : 1.f;
        const float sc = p.scale * g.step_mm * nm;
#pragma unroll
        for (int q = 0; q < FPT / 4; ++q) {
            const float4 yv = __ldg(reinterpret_cast<const float4 *>(p.yi + oy) + q);
            float4 rv;
            if (p.r_mode == KCS_R_PER_FRAME)
                rv = __ldg(reinterpret_cast<const float4 *>(p.r_pad + fg * FPT) + q);
            else
                rv = __ldg(reinterpret_cast<const float4 *>(p.ri + oy) + q);
            float4 out;
            float yh;
            yh = fmaf(sc, acc[4 * q + 0], rv.x); out.x = yh > 1e-12f ? nm * yv.x / yh : 0.f;
            yh = fmaf(sc, acc[4 * q + 1], rv.y); out.y = yh > 1e-12f ? nm * yv.y / yh : 0.f;
            yh = fmaf(sc, acc[4 * q + 2], rv.z); out.z = yh > 1e-12f ? nm * yv.z / yh : 0.f;
            yh = fmaf(sc, acc[4 * q + 3], rv.w); out.w = yh > 1e-12f ? nm * yv.w / yh : 0.f;
            reinterpret_cast<float4 *>(p.qi + o)[q] = out;
        }
    }
}

int kcs_launch_forward(kcs_ctx *c, int Tp, int subset, int ratio, float scale, int r_mode, int clip_fov, int z0, int nzc) {
    KGeom g = c->g;
    if (nzc <= 0) return KCS_OK;
    g.nz = nzc;  // slices [z0, z0 + nzc): direct planes are independent, a z range is a smaller problem of the same kind
    FwdArgs p;
    p.Tp = Tp;
    const int FPT = 4;  // one LDG.128 per lane and tap
    p.FG = Tp / FPT;
    p.As = subset < 0 ? g.A : g.A / g.S;
    p.xi = c->xi + (size_t)z0 * g.nyp * g.nxp * Tp;
    p.qi = c->qi + (size_t)z0 * p.As * g.B * Tp;
    p.yi = c->yi + (size_t)z0 * g.A * g.B * Tp;
    p.ri = c->ri ? c->ri + (size_t)z0 * g.A * g.B * Tp : nullptr;
    p.r_pad = c->r_pad;
    p.mult = (ratio && c->d_mult) ? c->d_mult + (size_t)z0 * g.A * g.B : nullptr;
    p.subset = subset;
    p.ratio = ratio; p.r_mode = r_mode; p.scale = scale;
    p.clip_r2 = clip_fov ? c->fov_rc2 : -1.f;
    {   // fractional bits of the fixed-point sample coordinates: 1 sign + ceil(log2(max dim + 32)) integer bits
        int ib = 1;
        while ((1 << ib) < (g.nxp > g.nyp ? g.nxp : g.nyp) + 2 * KCS_ANCHOR) ++ib;
        p.FB = 31 - ib > 22 ? 22 : 31 - ib;
    }
    // parallelism: split the K steps of a ray over KSPLIT threads when there are too few rays to fill 148 SMs.  Decided on
    // the WHOLE volume, not on the z range of this launch: the split fixes the order of a ray's partial sums, and a chunked
    // pass (kcs_icm_run_host) must reproduce the unchunked one bit for bit.
    const long long base = (long long)c->g.nz * p.As * g.B * p.FG;
    int ks = 1;
    while (base * ks < 148LL * 2048 && ks < 8 && g.K / (ks * 2) >= 16) ks *= 2;
    p.KSPLIT = ks;
    p.KCH = (g.K + ks - 1) / ks;
    int bins = KCS_FWD_TPB / (p.FG * ks);
    if (bins < 1) bins = 1;
    if (bins > g.B) bins = g.B;
    p.BINS = bins;
    const int threads = p.FG * bins * ks;
    const size_t smem = ks > 1 ? (size_t)(ks - 1) * FPT * bins * p.FG * sizeof(float) : 0;
    dim3 grid((g.B + bins - 1) / bins, p.As, g.nz);
    ProfScope ps(c, KCS_K_FORWARD);
    switch (p.FG) {
        case 1: k_forward<1><<<grid, threads, smem, c->stream>>>(g, p); break;
        case 2: k_forward<2><<<grid, threads, smem, c->stream>>>(g, p); break;
        case 4: k_forward<4><<<grid, threads, smem, c->stream>>>(g, p); break;
        default: k_forward<8><<<grid, threads, smem, c->stream>>>(g, p); break;
    }
    LAUNCH_CHECK(c);
    return KCS_OK;
}

// ---------------------------------------------------------------------------------------------------------
// Gather back-projector  (P4: exact transpose)
//   For voxel (i,j) and angle a the lattice coordinates (fb, fk) of the voxel centre follow from the inverse of
//   the sample map; only samples b in rint(fb)+{-1,0,1}, k in rint(fk)+{-1,0,1} can lie inside the voxel's tent
//   support (kcs_create checks the geometry ratio that guarantees this).  w_b = sum_k tent(dx) tent(dy).
// ---------------------------------------------------------------------------------------------------------
// Tent weight with reading Q23: a sample within 1e-9 pixel of a pixel centre lies ON it, so the weight
// is exactly 1 there and exactly 0 on the neighbours one pixel away (at 0 and 90 degrees every sample is such a sample;
// without the snap the weight left on the neighbour is rounding residue of ~1e-14).
__device__ __forceinline__ double tent_q23(double d) {
    const double ad = fabs(d);
    return ad < 1e-9 ? 1.0 : (ad > 1.0 - 1e-9 ? 0.0 : 1.0 - ad);
}

// Evaluated in fp64 (a geometry-only table, built once per context): a weight at the edge of a tent is a difference
// 1 - |d| of nearly equal numbers, and at low counts a voxel's update can hinge on that one weight (every other bin it
// sees holds y = 0), so the weights must be accurate RELATIVE to themselves, not to 1.
__device__ __forceinline__ float4 voxel_angle_weights(const KGeom &g, int a, int i, int j) {
    const double4 q = g.bwd[a];
    const double4 fw = g.fwd[a];
    const double xc = (double)i - g.cx, yc = (double)j - g.cy;
    const double fb = fma(xc, q.x, fma(yc, q.y, g.cb));
    const double fk = fma(xc, q.z, fma(yc, q.w, g.ck));
    const double rb = rint(fb), rk = rint(fk);
    const double db0 = rb - fb, dk0 = rk - fk;
    const int b1 = (int)rb, k1 = (int)rk;
    double w[3] = {0.0, 0.0, 0.0};
#pragma unroll
    for (int sk = -1; sk <= 1; ++sk) {
        const int k = k1 + sk;
        const bool kvalid = (k >= 0) && (k < g.K);
        const double dk = dk0 + (double)sk;
#pragma unroll
        for (int sb = -1; sb <= 1; ++sb) {
            const double db = db0 + (double)sb;
            const double dx = fma(db, fw.x, dk * fw.y), dy = fma(db, fw.z, dk * fw.w);
            const double t = tent_q23(dx) * tent_q23(dy);
            w[sb + 1] += kvalid ? t : 0.0;
        }
    }
    // re-align to a base bin b0c in [0, B-3] so the three loads never leave the row
    const int b0 = b1 - 1;
    const int b0c = max(0, min(b0, g.B - 3));
    float wo[3];
#pragma unroll
    for (int r = 0; r < 3; ++r) {
        const int rr = b0c + r - b0;
        wo[r] = (float)((rr == 0) ? w[0] : (rr == 1) ? w[1] : (rr == 2) ? w[2] : 0.0);
    }
    return make_float4(__int_as_float(b0c), wo[0], wo[1], wo[2]);
}

// O2 / eq. 2-3 with Q7-Q10, one division:  x bp / max(S (1 + beta (x-F)/Fm), 0.1 S)  with Fm = max(F, 1e-20)
//   = x bp Fm / (S max(Fm + beta (x-F), 0.1 Fm)).
__device__ __forceinline__ float osl_one(float x, float bp, float F, float S, float beta) {
    const float Fm = fmaxf(F, 1e-20f);
    const float den = S * fmaxf(fmaf(beta, x - F, Fm), 0.1f * Fm);
    return __fdividef(x * bp * Fm, den);
}

struct BackArgs {
    const float *qi;
    float *out;          // padded inner layout (plain back-projection) or xi (OSL, in place)
    const float *Fi;
    const float *sens;   // [ny][nx] unscaled A_s^T 1 of this subset, or [nz][ny][nx] unscaled A_s^T n (sens_z = 1)
    int sens_z;
    const float *smax;   // device scalar: max(sens)
    const unsigned char *mask;
    const float4 *wtab;  // [A][nbj][nbi4][KCS_BW][4] block-angle weight records (k_build_wtab)
    int nbj, nbi4;
    int Tp, FG, BX, BY, As, subset, osl;  // BX x BY blocks of 2x2 voxels per CTA
    float scale, beta;
};

#define KCS_BW 6  // float4 per (block, angle) weight record: {base bin, w[4 voxels][5 bins], pad}

// Geometry-only table, built once per context: for every angle a and every 2x2 voxel block (bi, bj) the base bin of the
// block's 5-bin window and the 4 x 5 tent weights (zero where a voxel does not see a bin; P4 / SURVEY H2).  Records of
// 4 x-adjacent blocks are interleaved float4-wise so that a warp's request for record word r is one 64 B run.
__global__ void k_build_wtab(KGeom g, float4 *wtab, int nbi, int nbj, int nbi4) {
    const int bi = blockIdx.x * blockDim.x + threadIdx.x;
    const int bj = blockIdx.y, a = blockIdx.z;
    if (bi >= nbi4 * 4) return;
    float4 w4[4];
    int bmin = 1 << 30;
#pragma unroll
    for (int v = 0; v < 4; ++v) {
        const int vi = 2 * bi + (v & 1), vj = 2 * bj + (v >> 1);
        if (bi < nbi && vi < g.nx && vj < g.ny) {
            w4[v] = voxel_angle_weights(g, a, vi, vj);  // {b0c, w0, w1, w2}, b0c in [0, B-3]
            bmin = min(bmin, __float_as_int(w4[v].x));
        } else {
            w4[v] = make_float4(__int_as_float(1 << 30), 0.f, 0.f, 0.f);
        }
    }
    const int base = max(0, min(bmin, g.B - 5));
    float w[4][5];
#pragma unroll
    for (int v = 0; v < 4; ++v) {
        const int sh = __float_as_int(w4[v].x) - base;  // 0..2 for an in-image voxel
#pragma unroll
        for (int r = 0; r < 5; ++r) {
            const int q = r - sh;
            w[v][r] = (q == 0) ? w4[v].y : (q == 1) ? w4[v].z : (q == 2) ? w4[v].w : 0.f;
        }
    }
    float4 *rec = wtab + (((size_t)a * nbj + bj) * nbi4 + (bi >> 2)) * (KCS_BW * 4) + (bi & 3);
    rec[0] = make_float4(__int_as_float(base), w[0][0], w[0][1], w[0][2]);
    rec[4] = make_float4(w[0][3], w[0][4], w[1][0], w[1][1]);
    rec[8] = make_float4(w[1][2], w[1][3], w[1][4], w[2][0]);
    rec[12] = make_float4(w[2][1], w[2][2], w[2][3], w[2][4]);
    rec[16] = make_float4(w[3][0], w[3][1], w[3][2], w[3][3]);
    rec[20] = make_float4(w[3][4], 0.f, 0.f, 0.f);
}

int kcs_launch_build_wtab(kcs_ctx *c) {
    const KGeom &g = c->g;
    dim3 grid((c->nbi4 * 4 + 63) / 64, c->nbj, g.A);
    ProfScope ps(c, KCS_K_OTHER);
    k_build_wtab<<<grid, 64, 0, c->stream>>>(g, c->d_wtab, c->nbi, c->nbj, c->nbi4);
    LAUNCH_CHECK(c);
    return KCS_OK;
}

// One thread = one 2x2 voxel block x 4 frames x ZB slices.  The four voxels of a block see bins inside one window of
// 5 consecutive bins (kcs_create guarantees (|cos| vx + |sin| vy)/bin <= 1.5, so their centre bins differ by <= 2):
// the window's 5 sinogram values are loaded once (5 LDG.128, one 128 B line each at Tp = 32) and serve all four
// voxels: 1.25 L1 wavefronts per voxel-angle instead of 3.  Weights come from the k_build_wtab table (L2 resident:
// it is the same for every slice and frame).  No atomics: run-to-run deterministic.
// Two instantiations are used (round 2, C4, per subset launch; results are bit-identical):
//   <2, true, .>   two slices per thread, the record of angle l+1 requested before the math of angle l, 4 CTAs per SM: the
//               plain back-projection (all 252 angles: 47.7 ms against 54.3);
//   <1, false, .>  one slice per thread, no prefetch, 80 registers, 6 CTAs per SM: the fused OSL update, whose epilogue
//               (x and F from HBM) overlaps other CTAs' angle loops better at 24 warps per SM (2.50 ms against 2.64).
// TPC: the padded frame count as a compile-time constant (32 on the ICM path of C2-C4: the window loads then take immediate
// offsets) or 0 for "read p.Tp".  Record and row pointers advance by constant strides from angle to angle; the loop body of
// <1, false, 32> went from 150 to 106 SASS instructions per angle for 80 FFMA with both.
template <int ZB, bool PIPE, int TPC>
__global__ void __launch_bounds__(KCS_BACK_TPB, PIPE ? 4 : 6) k_back(KGeom g, BackArgs p) {
    const int tid = threadIdx.x;
    const int fg = tid % p.FG;
    const int blk = tid / p.FG;
    const int bi = blockIdx.x * p.BX + blk % p.BX, bj = blockIdx.y * p.BY + blk / p.BX;
    const int i0 = bi * 2, j0 = bj * 2;
    const int z0 = blockIdx.z * ZB;
    const bool inimg = (i0 < g.nx) && (j0 < g.ny);
    bool vin[4], vact[4], active = false;
#pragma unroll
    for (int v = 0; v < 4; ++v) {
        const int i = i0 + (v & 1), j = j0 + (v >> 1);
        vin[v] = (i < g.nx) && (j < g.ny);
        vact[v] = vin[v] && (!p.osl || p.mask[j * g.nx + i] != 0);
        active = active || vact[v];
    }

    float acc[ZB][4][4];
#pragma unroll
    for (int zb = 0; zb < ZB; ++zb)
#pragma unroll
        for (int v = 0; v < 4; ++v)
#pragma unroll
            for (int f = 0; f < 4; ++f) acc[zb][v][f] = 0.f;

    const int Tp = TPC ? TPC : p.Tp;
    if (p.osl && active) {
        // the epilogue's x and F lines come from HBM (they do not fit L2 between subsets at C4): start them now
#pragma unroll
        for (int v = 0; v < 4; ++v) {
            if (!vact[v]) continue;
            const int i = i0 + (v & 1), j = j0 + (v >> 1);
#pragma unroll
            for (int zb = 0; zb < ZB; ++zb) {
                const int z = z0 + zb;
                if (z >= g.nz) break;
                const size_t o = (((size_t)z * g.nyp + (j + KCS_PAD)) * g.nxp + (i + KCS_PAD)) * Tp + fg * 4;
                asm volatile("prefetch.global.L2 [%0];" ::"l"(p.out + o));
                asm volatile("prefetch.global.L2 [%0];" ::"l"(p.Fi + o));
            }
        }
    }
    if (active) {
        const size_t astride = (size_t)p.nbj * p.nbi4 * (KCS_BW * 4);
        const float4 *rec0 = p.wtab + ((size_t)bj * p.nbi4 + (bi >> 2)) * (KCS_BW * 4) + (bi & 3);
        // Software pipeline: the record of angle l+1 is requested before the math of angle l, and the windows of all ZB
        // slices of an angle are requested together, so a thread waits on global memory once per angle, not ZB+1 times
        // (ncu source page of the un-pipelined loop: 16 % of the stall samples on the record, 4 x 5.5 % on the windows).
        const size_t rstep = (size_t)(p.subset < 0 ? 1 : g.S) * astride;          // record stride from angle to angle
        const float4 *rec = rec0 + (size_t)(p.subset < 0 ? 0 : p.subset) * astride;  // record of the angle to load next
        const size_t qstep = (size_t)g.B * Tp;                                      // sinogram row stride from angle to angle
        const float *ql[ZB];
#pragma unroll
        for (int zb = 0; zb < ZB; ++zb) {
            const int z = min(z0 + zb, g.nz - 1);  // a slice beyond the volume re-reads the last one; its result is dropped
            ql[zb] = p.qi + (size_t)z * p.As * qstep + fg * 4;
        }
        float4 n0, n1, n2, n3, n4, n5;
        if (PIPE) {
            n0 = __ldg(rec); n1 = __ldg(rec + 4); n2 = __ldg(rec + 8); n3 = __ldg(rec + 12); n4 = __ldg(rec + 16); n5 = __ldg(rec + 20);
            rec += rstep;
        }
        for (int l = 0; l < p.As; ++l) {
            if (!PIPE) {
                n0 = __ldg(rec); n1 = __ldg(rec + 4); n2 = __ldg(rec + 8); n3 = __ldg(rec + 12); n4 = __ldg(rec + 16); n5 = __ldg(rec + 20);
                rec += rstep;
            }
            const float4 r0 = n0, r1 = n1, r2 = n2, r3 = n3, r4 = n4, r5 = n5;
            const int base = __float_as_int(r0.x);
            float4 q[ZB][5];
#pragma unroll
            for (int zb = 0; zb < ZB; ++zb) {
                const float *row = ql[zb] + (size_t)base * Tp;
#pragma unroll
                for (int r = 0; r < 5; ++r) q[zb][r] = __ldg(reinterpret_cast<const float4 *>(row + r * Tp));
                ql[zb] += qstep;
            }
            if (PIPE && l + 1 < p.As) {
                n0 = __ldg(rec); n1 = __ldg(rec + 4); n2 = __ldg(rec + 8); n3 = __ldg(rec + 12); n4 = __ldg(rec + 16); n5 = __ldg(rec + 20);
                rec += rstep;
            }
            const float w[4][5] = {{r0.y, r0.z, r0.w, r1.x, r1.y},
                                   {r1.z, r1.w, r2.x, r2.y, r2.z},
                                   {r2.w, r3.x, r3.y, r3.z, r3.w},
                                   {r4.x, r4.y, r4.z, r4.w, r5.x}};
#pragma unroll
            for (int zb = 0; zb < ZB; ++zb) {
#pragma unroll
                for (int v = 0; v < 4; ++v) {
#pragma unroll
                    for (int r = 0; r < 5; ++r) {
                        acc[zb][v][0] = fmaf(w[v][r], q[zb][r].x, acc[zb][v][0]);
                        acc[zb][v][1] = fmaf(w[v][r], q[zb][r].y, acc[zb][v][1]);
                        acc[zb][v][2] = fmaf(w[v][r], q[zb][r].z, acc[zb][v][2]);
                        acc[zb][v][3] = fmaf(w[v][r], q[zb][r].w, acc[zb][v][3]);
                    }
                }
            }
        }
    }
    if (!inimg) return;

    if (!p.osl) {
#pragma unroll
        for (int v = 0; v < 4; ++v) {
            if (!vin[v]) continue;
            const int i = i0 + (v & 1), j = j0 + (v >> 1);
#pragma unroll
            for (int zb = 0; zb < ZB; ++zb) {
                const int z = z0 + zb;
                if (z >= g.nz) break;
                const size_t o = (((size_t)z * g.nyp + (j + KCS_PAD)) * g.nxp + (i + KCS_PAD)) * Tp + fg * 4;
                *reinterpret_cast<float4 *>(p.out + o) = make_float4(g.step_mm * acc[zb][v][0], g.step_mm * acc[zb][v][1],
                                                                     g.step_mm * acc[zb][v][2], g.step_mm * acc[zb][v][3]);
            }
        }
        return;
    }
    // O2 / eq. 2-3 with Q7-Q10:  x <- x * bp / max(S (1 + beta (x-F)/max(F,1e-20)), 0.1 S).  All x and F lines of the
    // thread are requested first (they come from L2 / HBM), then updated and stored: one wait instead of 4 ZB.
    const float smax = *p.smax;
    const float sc = p.scale * g.step_mm;
    const size_t v2 = (size_t)g.nx * g.ny;
    float4 xv[4][ZB], Fv[4][ZB];
    float Sv[4][ZB];
    bool live[4][ZB];
#pragma unroll
    for (int v = 0; v < 4; ++v) {
        const int i = min(i0 + (v & 1), g.nx - 1), j = min(j0 + (v >> 1), g.ny - 1);
#pragma unroll
        for (int zb = 0; zb < ZB; ++zb) {
            const int z = min(z0 + zb, g.nz - 1);
            const float S0 = p.sens[(p.sens_z ? (size_t)z * v2 : 0) + (size_t)j * g.nx + i];
            Sv[v][zb] = p.scale * S0;
            live[v][zb] = vact[v] && (S0 > 1e-12f * smax);
            const size_t o = (((size_t)z * g.nyp + (j + KCS_PAD)) * g.nxp + (i + KCS_PAD)) * Tp + fg * 4;
            xv[v][zb] = make_float4(0.f, 0.f, 0.f, 0.f);
            Fv[v][zb] = make_float4(1.f, 1.f, 1.f, 1.f);
            if (live[v][zb]) {
                xv[v][zb] = *reinterpret_cast<const float4 *>(p.out + o);
                Fv[v][zb] = __ldg(reinterpret_cast<const float4 *>(p.Fi + o));
            }
        }
    }
#pragma unroll
    for (int v = 0; v < 4; ++v) {
        if (!vin[v]) continue;
        const int i = i0 + (v & 1), j = j0 + (v >> 1);
#pragma unroll
        for (int zb = 0; zb < ZB; ++zb) {
            const int z = z0 + zb;
            if (z >= g.nz) break;
            const size_t o = (((size_t)z * g.nyp + (j + KCS_PAD)) * g.nxp + (i + KCS_PAD)) * Tp + fg * 4;
            float4 out = make_float4(0.f, 0.f, 0.f, 0.f);  // outside the mask or without sensitivity: x = 0 (Q2, Q10)
            if (live[v][zb]) {
                out.x = osl_one(xv[v][zb].x, sc * acc[zb][v][0], Fv[v][zb].x, Sv[v][zb], p.beta);
                out.y = osl_one(xv[v][zb].y, sc * acc[zb][v][1], Fv[v][zb].y, Sv[v][zb], p.beta);
                out.z = osl_one(xv[v][zb].z, sc * acc[zb][v][2], Fv[v][zb].z, Sv[v][zb], p.beta);
                out.w = osl_one(xv[v][zb].w, sc * acc[zb][v][3], Fv[v][zb].w, Sv[v][zb], p.beta);
            }
            *reinterpret_cast<float4 *>(p.out + o) = out;
        }
    }
}

int kcs_launch_back(kcs_ctx *c, int Tp, int subset, int osl, float *out_inner, float scale, float beta, int z0, int nzc) {
    KGeom g = c->g;
    if (nzc <= 0) return KCS_OK;
    g.nz = nzc;  // slices [z0, z0 + nzc)
    BackArgs p;
    const size_t zpix = (size_t)z0 * g.nyp * g.nxp * Tp;
    p.qi = c->qi + (size_t)z0 * (subset < 0 ? g.A : g.A / g.S) * g.B * Tp;
    p.out = (osl ? c->xi : out_inner) + zpix;
    p.Fi = c->Fi + zpix;
    const int sidx = subset < 0 ? g.S : subset;
    p.sens_z = (osl && c->d_mult && subset >= 0) ? 1 : 0;
    if (p.sens_z) {  // S8(f)3: A_s^T n differs from slice to slice
        p.sens = c->d_sens_z + ((size_t)subset * c->g.nz + z0) * g.nx * g.ny;
        p.smax = c->d_smax_z + subset;
    } else {
        p.sens = c->d_sens + (size_t)sidx * g.nx * g.ny;
        p.smax = c->d_smax + sidx;
    }
    p.mask = c->d_mask;
    p.Tp = Tp;
    p.FG = Tp / 4;
    p.As = subset < 0 ? g.A : g.A / g.S;
    p.subset = subset;
    p.osl = osl; p.scale = scale; p.beta = beta;
    p.wtab = c->d_wtab; p.nbj = c->nbj; p.nbi4 = c->nbi4;
    const int nblk = KCS_BACK_TPB / p.FG;        // 16 .. 128 voxel blocks per CTA
    p.BX = nblk >= 128 ? 16 : 8;
    p.BY = nblk / p.BX;
    const int gx = (g.nx + 2 * p.BX - 1) / (2 * p.BX), gy = (g.ny + 2 * p.BY - 1) / (2 * p.BY);
    // plain back-projection: two slices per thread when that still fills the GPU; fused OSL update: one (see k_back)
    int ZB = 1;
    if (!osl && g.nz >= 2 && (long long)gx * gy * ((g.nz + 1) / 2) >= 148LL) ZB = 2;
    dim3 grid(gx, gy, (g.nz + ZB - 1) / ZB);
    ProfScope ps(c, KCS_K_BACK);
    if (osl && Tp == 32) k_back<1, false, 32><<<grid, KCS_BACK_TPB, 0, c->stream>>>(g, p);
    else if (osl) k_back<1, false, 0><<<grid, KCS_BACK_TPB, 0, c->stream>>>(g, p);
    else if (ZB == 2 && Tp == 32) k_back<2, true, 32><<<grid, KCS_BACK_TPB, 0, c->stream>>>(g, p);
    else if (ZB == 2) k_back<2, true, 0><<<grid, KCS_BACK_TPB, 0, c->stream>>>(g, p);
    else k_back<1, true, 0><<<grid, KCS_BACK_TPB, 0, c->stream>>>(g, p);
    LAUNCH_CHECK(c);
    return KCS_OK;
}

// ---------------------------------------------------------------------------------------------------------
// Sensitivity images A_s^T 1 (one slice, all subsets + all-angle image) and their maxima.
// ---------------------------------------------------------------------------------------------------------
__global__ void k_sens(KGeom g, float *sens, float *smax) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y;
    const int s = blockIdx.z;  // s == S: all angles
    if (i >= g.nx) return;
    const int As = s == g.S ? g.A : g.A / g.S;
    double acc = 0.0;
    for (int la = 0; la < As; ++la) {
        const int a = s == g.S ? la : s + la * g.S;
        const float4 w = voxel_angle_weights(g, a, i, j);
        acc += (double)w.y + (double)w.z + (double)w.w;
    }
    const float sum = (float)(acc * (double)g.step_mm);
    sens[((size_t)s * g.ny + j) * g.nx + i] = sum;
    atomicMax(reinterpret_cast<int *>(smax + s), __float_as_int(sum));  // sum >= 0: int order == float order
}

int kcs_launch_sens(kcs_ctx *c) {
    const KGeom &g = c->g;
    cudaError_t e = cudaMemsetAsync(c->d_smax, 0, sizeof(float) * (g.S + 1), c->stream);
    if (e != cudaSuccess) { c->err = cudaGetErrorString(e); return KCS_ERR_CUDA; }
    dim3 grid((g.nx + 127) / 128, g.ny, g.S + 1);
    ProfScope ps(c, KCS_K_OTHER);
    k_sens<<<grid, 128, 0, c->stream>>>(g, c->d_sens, c->d_smax);
    LAUNCH_CHECK(c);
    return KCS_OK;
}

// ---------------------------------------------------------------------------------------------------------
// Stand-alone OSL update on planar buffers (kcs_osl_update).
// ---------------------------------------------------------------------------------------------------------
__global__ void k_max_nonneg(const float *v, size_t n, float *out) {
    float m = 0.f;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < n; q += (size_t)gridDim.x * blockDim.x) m = fmaxf(m, v[q]);
    for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) atomicMax(reinterpret_cast<int *>(out), __float_as_int(fmaxf(m, 0.f)));
}

__global__ void k_osl_planar(float *x, const float *bp, const float *sens, const float *F, const unsigned char *mask,
                             const float *smax, size_t n, int v2, float beta, int prior_mode, float sigma2) {
    const size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= n) return;
    const int pix = (int)(q % (size_t)v2);
    const float S = sens[pix];
    if (!mask[pix] || !(S > 1e-12f * *smax)) {
        x[q] = 0.f;
        return;
    }
    const float xv = x[q], Fv = F[q];
    float D;
    if (prior_mode == KCS_PRIOR_POISSON_MATCHED)
        D = S * (1.f + beta * (xv - Fv) / fmaxf(Fv, 1e-20f));
    else
        D = S + beta * (xv - Fv) / sigma2;
    D = fmaxf(D, 0.1f * S);
    x[q] = xv * bp[q] / D;
}

// n[nz][A][B] restricted to the angles of one subset: out[z][la][b] = n[z][s + la S][b]  (one frame of a subset sinogram)
__global__ void k_subset_rows(const float *__restrict__ n, float *__restrict__ out, int nz, int A, int B, int S, int s) {
    const int As = A / S;
    const size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= (size_t)nz * As * B) return;
    const int b = (int)(q % B), la = (int)((q / B) % As), z = (int)(q / ((size_t)B * As));
    out[q] = n[((size_t)z * A + (s + la * S)) * B + b];
}

int kcs_launch_subset_rows(kcs_ctx *c, const float *n, float *out, int s) {
    const KGeom &g = c->g;
    const size_t tot = (size_t)g.nz * (g.A / g.S) * g.B;
    ProfScope ps(c, KCS_K_OTHER);
    k_subset_rows<<<(unsigned)((tot + 255) / 256), 256, 0, c->stream>>>(n, out, g.nz, g.A, g.B, g.S, s);
    LAUNCH_CHECK(c);
    return KCS_OK;
}

int kcs_launch_max_nonneg(kcs_ctx *c, const float *v, size_t n, float *out) {
    cudaError_t e = cudaMemsetAsync(out, 0, sizeof(float), c->stream);
    if (e != cudaSuccess) { c->err = cudaGetErrorString(e); return KCS_ERR_CUDA; }
    ProfScope ps(c, KCS_K_OTHER);
    k_max_nonneg<<<256, 256, 0, c->stream>>>(v, n, out);
    LAUNCH_CHECK(c);
    return KCS_OK;
}

int kcs_launch_osl_planar(kcs_ctx *c, float *x, const float *bp, const float *sens, const float *F, float beta,
                          int prior_mode, float sigma2) {
    const KGeom &g = c->g;
    const int v2 = g.nx * g.ny;
    cudaError_t e = cudaMemsetAsync(c->d_tmp_smax, 0, sizeof(float), c->stream);
    if (e != cudaSuccess) { c->err = cudaGetErrorString(e); return KCS_ERR_CUDA; }
    ProfScope ps(c, KCS_K_OTHER);
    k_max_nonneg<<<64, 256, 0, c->stream>>>(sens, (size_t)v2, c->d_tmp_smax);
    LAUNCH_CHECK(c);
    const size_t n = (size_t)c->cfg.n_frames * c->n_vox;
    k_osl_planar<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(x, bp, sens, F, c->d_mask, c->d_tmp_smax, n, v2, beta,
                                                                     prior_mode, sigma2);
    LAUNCH_CHECK(c);
    return KCS_OK;
}
