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

__device__ __forceinline__ long long pack_dst(const PackMap &m, long long row, int col) {
    return (row / m.rps) * m.slab + (long long)(row % m.rps) * m.rstride + m.off + col;
}

// block (32, 8): one row segment of 32 columns, all frames.
__global__ void k_pack(const float *__restrict__ src, size_t fs, int nf, float *__restrict__ dst, int Tp, PackMap m) {
    __shared__ float tile[KCS_MAX_FRAMES][33];
    const int c0 = blockIdx.x * 32;
    const long long row = blockIdx.y + (long long)blockIdx.z * gridDim.y;
    if (row >= m.nrows) return;
    const int tx = threadIdx.x, ty = threadIdx.y;
    for (int f = ty; f < Tp; f += 8) {
        float v = 0.f;
        if (f < nf && c0 + tx < m.W) v = src[(size_t)f * fs + (size_t)row * m.W + c0 + tx];
        tile[f][tx] = v;
    }
    __syncthreads();
    const int ncol = min(32, m.W - c0);
    const long long d0 = pack_dst(m, row, c0);
    const int n = ncol * Tp;
    for (int e = ty * 32 + tx; e < n; e += 256) {
        const int col = e / Tp, f = e - col * Tp;
        dst[(size_t)d0 * Tp + e] = tile[f][col];
    }
}

__global__ void k_unpack(const float *__restrict__ src, int Tp, float *__restrict__ dst, size_t fs, int nf, PackMap m) {
    __shared__ float tile[KCS_MAX_FRAMES][33];
    const int c0 = blockIdx.x * 32;
    const long long row = blockIdx.y + (long long)blockIdx.z * gridDim.y;
    if (row >= m.nrows) return;
    const int tx = threadIdx.x, ty = threadIdx.y;
    const int ncol = min(32, m.W - c0);
    const long long d0 = pack_dst(m, row, c0);
    const int n = ncol * Tp;
    for (int e = ty * 32 + tx; e < n; e += 256) {
        const int col = e / Tp, f = e - col * Tp;
        tile[f][col] = src[(size_t)d0 * Tp + e];
    }
    __syncthreads();
    for (int f = ty; f < nf; f += 8)
        if (c0 + tx < m.W) dst[(size_t)f * fs + (size_t)row * m.W + c0 + tx] = tile[f][tx];
}

static void pack_grid(long long nrows, int W, dim3 &grid) {
    const long long gy = nrows < 32768 ? nrows : 32768;
    grid = dim3((unsigned)((W + 31) / 32), (unsigned)gy, (unsigned)((nrows + gy - 1) / gy));
}

int kcs_launch_pack(kcs_ctx *c, const float *src, size_t fs, int nf, float *dst, int Tp, long long nrows, int W,
                    int rps, long long slab, int rstride, int off) {
    PackMap m{nrows, W, rps, slab, rstride, off};
    dim3 grid;
    pack_grid(nrows, W, grid);
    ProfScope ps(c, KCS_K_PACK);
    k_pack<<<grid, dim3(32, 8), 0, c->stream>>>(src, fs, nf, dst, Tp, m);
    LAUNCH_CHECK(c);
    return KCS_OK;
}

int kcs_launch_unpack(kcs_ctx *c, const float *src, int Tp, float *dst, size_t fs, int nf, long long nrows, int W,
                      int rps, long long slab, int rstride, int off) {
    PackMap m{nrows, W, rps, slab, rstride, off};
    dim3 grid;
    pack_grid(nrows, W, grid);
    ProfScope ps(c, KCS_K_UNPACK);
    k_unpack<<<grid, dim3(32, 8), 0, c->stream>>>(src, Tp, dst, fs, nf, m);
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
    int Tp, FG, BINS, KSPLIT, KCH;
    int As, subset;
    int ratio, r_mode;
    float scale;
};

#define KCS_ANCHOR 16  // steps between fp64 re-anchoring of the sample coordinates

template <int FPT>
__global__ void __launch_bounds__(256) k_forward(KGeom g, FwdArgs p) {
    extern __shared__ float red[];
    const int tid = threadIdx.x;
    const int fg = tid % p.FG;
    const int bl = (tid / p.FG) % p.BINS;
    const int kc = tid / (p.FG * p.BINS);
    const int b = blockIdx.x * p.BINS + bl;
    const int la = blockIdx.y, z = blockIdx.z;
    const int a = p.subset < 0 ? la : p.subset + la * g.S;

    float acc[FPT];
#pragma unroll
    for (int f = 0; f < FPT; ++f) acc[f] = 0.f;

    if (b < g.B) {
        const double4 fw = g.fwd[a];
        const double bc = (double)b - g.cb;
        const float dxk = (float)fw.y, dyk = (float)fw.w;
        const int k_lo = kc * p.KCH;
        const int k_hi = min(g.K, k_lo + p.KCH);
        const int Tp = p.Tp;
        const int rowstride = g.nxp * Tp;
        const float *slice = p.xi + (size_t)z * g.nyp * rowstride + fg * FPT;
        for (int k0 = k_lo; k0 < k_hi; k0 += KCS_ANCHOR) {
            // fp64 anchor (P2): padded continuous index of sample (b, k0); integer part kept as int, fraction as fp32
            const double kk = (double)k0 - g.ck;
            const double px0 = fma(kk, fw.y, fma(bc, fw.x, g.cx + 1.0));
            const double py0 = fma(kk, fw.w, fma(bc, fw.z, g.cy + 1.0));
            const double flx0 = floor(px0), fly0 = floor(py0);
            const int ia = (int)flx0, ja = (int)fly0;
            const float fax = (float)(px0 - flx0), fay = (float)(py0 - fly0);
            const int mmax = min(KCS_ANCHOR, k_hi - k0);
            for (int m = 0; m < mmax; ++m) {
                const float fxm = fmaf((float)m, dxk, fax), fym = fmaf((float)m, dyk, fay);
                const float flx = floorf(fxm), fly = floorf(fym);
                const float wx = fxm - flx, wy = fym - fly;
                const int i0 = ia + (int)flx, j0 = ja + (int)fly;
                if ((unsigned)i0 <= (unsigned)g.nx && (unsigned)j0 <= (unsigned)g.ny) {
                    const float *p00 = slice + (size_t)j0 * rowstride + i0 * Tp;
                    const float w00 = (1.f - wx) * (1.f - wy), w10 = wx * (1.f - wy);
                    const float w01 = (1.f - wx) * wy, w11 = wx * wy;
#pragma unroll
                    for (int q = 0; q < FPT / 4; ++q) {
                        const float4 v00 = __ldg(reinterpret_cast<const float4 *>(p00) + q);
                        const float4 v10 = __ldg(reinterpret_cast<const float4 *>(p00 + Tp) + q);
                        const float4 v01 = __ldg(reinterpret_cast<const float4 *>(p00 + rowstride) + q);
                        const float4 v11 = __ldg(reinterpret_cast<const float4 *>(p00 + rowstride + Tp) + q);
                        acc[4 * q + 0] += w00 * v00.x + w10 * v10.x + w01 * v01.x + w11 * v11.x;
                        acc[4 * q + 1] += w00 * v00.y + w10 * v10.y + w01 * v01.y + w11 * v11.y;
                        acc[4 * q + 2] += w00 * v00.z + w10 * v10.z + w01 * v01.z + w11 * v11.z;
                        acc[4 * q + 3] += w00 * v00.w + w10 * v10.w + w01 * v01.w + w11 * v11.w;
                    }
                }
            }
        }
    }

    // combine the KSPLIT partial sums of a ray (fixed order: deterministic)
    if (p.KSPLIT > 1) {
        const int nbf = p.BINS * p.FG;
        const int idx = bl * p.FG + fg;
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

    const size_t o = (((size_t)z * p.As + la) * g.B + b) * p.Tp + fg * FPT;
    if (!p.ratio) {
#pragma unroll
        for (int q = 0; q < FPT / 4; ++q)
            reinterpret_cast<float4 *>(p.qi + o)[q] = make_float4(g.step_mm * acc[4 * q], g.step_mm * acc[4 * q + 1],
                                                                  g.step_mm * acc[4 * q + 2], g.step_mm * acc[4 * q + 3]);
    } else {
        // O1: yhat = scale A_s x + r ; q = y / yhat where yhat > 1e-12 else 0
        const size_t oy = (((size_t)z * g.A + a) * g.B + b) * p.Tp + fg * FPT;
        const float sc = p.scale * g.step_mm;
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
            yh = fmaf(sc, acc[4 * q + 0], rv.x); out.x = yh > 1e-12f ? yv.x / yh : 0.f;
            yh = fmaf(sc, acc[4 * q + 1], rv.y); out.y = yh > 1e-12f ? yv.y / yh : 0.f;
            yh = fmaf(sc, acc[4 * q + 2], rv.z); out.z = yh > 1e-12f ? yv.z / yh : 0.f;
            yh = fmaf(sc, acc[4 * q + 3], rv.w); out.w = yh > 1e-12f ? yv.w / yh : 0.f;
            reinterpret_cast<float4 *>(p.qi + o)[q] = out;
        }
    }
}

int kcs_launch_forward(kcs_ctx *c, int Tp, int subset, int ratio, float scale, int r_mode) {
    const KGeom &g = c->g;
    FwdArgs p;
    p.xi = c->xi; p.qi = c->qi; p.yi = c->yi; p.ri = c->ri; p.r_pad = c->r_pad;
    p.Tp = Tp;
    const int FPT = choose_fpt(Tp);
    p.FG = Tp / FPT;
    p.As = subset < 0 ? g.A : g.A / g.S;
    p.subset = subset;
    p.ratio = ratio; p.r_mode = r_mode; p.scale = scale;
    // parallelism: split the K steps of a ray over KSPLIT threads when there are too few rays to fill 148 SMs
    const long long base = (long long)g.nz * p.As * g.B * p.FG;
    int ks = 1;
    while (base * ks < 148LL * 2048 && ks < 8 && g.K / (ks * 2) >= 16) ks *= 2;
    p.KSPLIT = ks;
    p.KCH = (g.K + ks - 1) / ks;
    int bins = 128 / (p.FG * ks);
    if (bins < 1) bins = 1;
    if (bins > g.B) bins = g.B;
    p.BINS = bins;
    const int threads = p.FG * bins * ks;
    const size_t smem = ks > 1 ? (size_t)(ks - 1) * FPT * bins * p.FG * sizeof(float) : 0;
    dim3 grid((g.B + bins - 1) / bins, p.As, g.nz);
    ProfScope ps(c, KCS_K_FORWARD);
    switch (FPT) {
        case 4: k_forward<4><<<grid, threads, smem, c->stream>>>(g, p); break;
        case 8: k_forward<8><<<grid, threads, smem, c->stream>>>(g, p); break;
        default: k_forward<12><<<grid, threads, smem, c->stream>>>(g, p); break;
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
__device__ __forceinline__ float4 voxel_angle_weights(const KGeom &g, int a, int i, int j) {
    const double4 q = g.bwd[a];
    const double4 fw = g.fwd[a];
    const double xc = (double)i - g.cx, yc = (double)j - g.cy;
    const double fb = fma(xc, q.x, fma(yc, q.y, g.cb));
    const double fk = fma(xc, q.z, fma(yc, q.w, g.ck));
    const double rb = rint(fb), rk = rint(fk);
    const float db0 = (float)(rb - fb), dk0 = (float)(rk - fk);
    const int b1 = (int)rb, k1 = (int)rk;
    const float axb = (float)fw.x, axk = (float)fw.y, ayb = (float)fw.z, ayk = (float)fw.w;
    float w[3] = {0.f, 0.f, 0.f};
#pragma unroll
    for (int sk = -1; sk <= 1; ++sk) {
        const int k = k1 + sk;
        const bool kvalid = (k >= 0) && (k < g.K);
        const float dk = dk0 + (float)sk;
#pragma unroll
        for (int sb = -1; sb <= 1; ++sb) {
            const float db = db0 + (float)sb;
            const float dx = fmaf(db, axb, dk * axk), dy = fmaf(db, ayb, dk * ayk);
            const float t = fmaxf(0.f, 1.f - fabsf(dx)) * fmaxf(0.f, 1.f - fabsf(dy));
            w[sb + 1] += kvalid ? t : 0.f;
        }
    }
    // re-align to a base bin b0c in [0, B-3] so the three loads never leave the row
    const int b0 = b1 - 1;
    const int b0c = max(0, min(b0, g.B - 3));
    float wo[3];
#pragma unroll
    for (int r = 0; r < 3; ++r) {
        const int rr = b0c + r - b0;
        wo[r] = (rr == 0) ? w[0] : (rr == 1) ? w[1] : (rr == 2) ? w[2] : 0.f;
    }
    return make_float4(__int_as_float(b0c), wo[0], wo[1], wo[2]);
}

struct BackArgs {
    const float *qi;
    float *out;          // padded inner layout (plain back-projection) or xi (OSL, in place)
    const float *Fi;
    const float *sens;   // [ny][nx] unscaled A_s^T 1 of this subset
    const float *smax;   // device scalar: max(sens)
    const unsigned char *mask;
    int Tp, FG, TX, TY, As, subset, osl;
    float scale, beta;
};

#define KCS_BACK_ACH 16  // angles per shared-memory weight chunk

template <int FPT, int ZB>
__global__ void __launch_bounds__(256) k_back(KGeom g, BackArgs p) {
    extern __shared__ float4 wts[];  // [KCS_BACK_ACH][NVOX]
    const int tid = threadIdx.x;
    const int nvox = p.TX * p.TY;
    const int fg = tid % p.FG;
    const int vox = tid / p.FG;
    const int i = blockIdx.x * p.TX + vox % p.TX;
    const int j = blockIdx.y * p.TY + vox / p.TX;
    const int z0 = blockIdx.z * ZB;
    const bool inimg = (vox < nvox) && (i < g.nx) && (j < g.ny);
    bool active = inimg;
    if (p.osl && inimg) active = p.mask[j * g.nx + i] != 0;

    float acc[ZB][FPT];
#pragma unroll
    for (int zb = 0; zb < ZB; ++zb)
#pragma unroll
        for (int f = 0; f < FPT; ++f) acc[zb][f] = 0.f;

    const int Tp = p.Tp;
    for (int la0 = 0; la0 < p.As; la0 += KCS_BACK_ACH) {
        const int nla = min(KCS_BACK_ACH, p.As - la0);
        __syncthreads();
        for (int item = tid; item < nla * nvox; item += blockDim.x) {
            const int l = item / nvox, v = item - l * nvox;
            const int vi = blockIdx.x * p.TX + v % p.TX, vj = blockIdx.y * p.TY + v / p.TX;
            const int a = p.subset < 0 ? (la0 + l) : p.subset + (la0 + l) * g.S;
            wts[item] = voxel_angle_weights(g, a, vi, vj);
        }
        __syncthreads();
        if (active) {
            for (int l = 0; l < nla; ++l) {
                const float4 w = wts[l * nvox + vox];
                const int b0 = __float_as_int(w.x);
#pragma unroll
                for (int zb = 0; zb < ZB; ++zb) {
                    const int z = z0 + zb;
                    if (z < g.nz) {
                        const float *row = p.qi + (((size_t)z * p.As + (la0 + l)) * g.B + b0) * Tp + fg * FPT;
#pragma unroll
                        for (int q = 0; q < FPT / 4; ++q) {
                            const float4 q0 = __ldg(reinterpret_cast<const float4 *>(row) + q);
                            const float4 q1 = __ldg(reinterpret_cast<const float4 *>(row + Tp) + q);
                            const float4 q2 = __ldg(reinterpret_cast<const float4 *>(row + 2 * Tp) + q);
                            acc[zb][4 * q + 0] += w.y * q0.x + w.z * q1.x + w.w * q2.x;
                            acc[zb][4 * q + 1] += w.y * q0.y + w.z * q1.y + w.w * q2.y;
                            acc[zb][4 * q + 2] += w.y * q0.z + w.z * q1.z + w.w * q2.z;
                            acc[zb][4 * q + 3] += w.y * q0.w + w.z * q1.w + w.w * q2.w;
                        }
                    }
                }
            }
        }
    }
    if (!inimg) return;

    const float S0 = p.osl ? p.sens[j * g.nx + i] : 0.f;
    const float smax = p.osl ? *p.smax : 0.f;
#pragma unroll
    for (int zb = 0; zb < ZB; ++zb) {
        const int z = z0 + zb;
        if (z >= g.nz) break;
        const size_t o = (((size_t)z * g.nyp + (j + 1)) * g.nxp + (i + 1)) * Tp + fg * FPT;
        if (!p.osl) {
#pragma unroll
            for (int q = 0; q < FPT / 4; ++q)
                reinterpret_cast<float4 *>(p.out + o)[q] =
                    make_float4(g.step_mm * acc[zb][4 * q], g.step_mm * acc[zb][4 * q + 1],
                                g.step_mm * acc[zb][4 * q + 2], g.step_mm * acc[zb][4 * q + 3]);
        } else {
            // O2 / eq. 2-3 with Q7-Q10:  x <- x * bp / max(S (1 + beta (x-F)/max(F,1e-20)), 0.1 S)
            const float S = p.scale * S0;
            const bool dead = (!active) || !(S0 > 1e-12f * smax);
            const float sc = p.scale * g.step_mm;
#pragma unroll
            for (int q = 0; q < FPT / 4; ++q) {
                float4 xv = reinterpret_cast<const float4 *>(p.out + o)[q];
                if (dead) {
                    xv = make_float4(0.f, 0.f, 0.f, 0.f);
                } else {
                    const float4 Fv = __ldg(reinterpret_cast<const float4 *>(p.Fi + o) + q);
                    float D;
                    D = S * (1.f + p.beta * (xv.x - Fv.x) / fmaxf(Fv.x, 1e-20f)); D = fmaxf(D, 0.1f * S);
                    xv.x = xv.x * (sc * acc[zb][4 * q + 0]) / D;
                    D = S * (1.f + p.beta * (xv.y - Fv.y) / fmaxf(Fv.y, 1e-20f)); D = fmaxf(D, 0.1f * S);
                    xv.y = xv.y * (sc * acc[zb][4 * q + 1]) / D;
                    D = S * (1.f + p.beta * (xv.z - Fv.z) / fmaxf(Fv.z, 1e-20f)); D = fmaxf(D, 0.1f * S);
                    xv.z = xv.z * (sc * acc[zb][4 * q + 2]) / D;
                    D = S * (1.f + p.beta * (xv.w - Fv.w) / fmaxf(Fv.w, 1e-20f)); D = fmaxf(D, 0.1f * S);
                    xv.w = xv.w * (sc * acc[zb][4 * q + 3]) / D;
                }
                reinterpret_cast<float4 *>(p.out + o)[q] = xv;
            }
        }
    }
}

template <int FPT>
static void back_dispatch(int ZB, dim3 grid, int threads, size_t smem, cudaStream_t st, const KGeom &g, const BackArgs &p) {
    static bool optin = false;  // the weight chunk can exceed the 48 KB default (64 KB at 256 voxels per block)
    if (!optin) {
        cudaFuncSetAttribute(k_back<FPT, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024);
        cudaFuncSetAttribute(k_back<FPT, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024);
        cudaFuncSetAttribute(k_back<FPT, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024);
        optin = true;
    }
    switch (ZB) {
        case 4: k_back<FPT, 4><<<grid, threads, smem, st>>>(g, p); break;
        case 2: k_back<FPT, 2><<<grid, threads, smem, st>>>(g, p); break;
        default: k_back<FPT, 1><<<grid, threads, smem, st>>>(g, p); break;
    }
}

int kcs_launch_back(kcs_ctx *c, int Tp, int subset, int osl, float *out_inner, float scale, float beta) {
    const KGeom &g = c->g;
    BackArgs p;
    p.qi = c->qi;
    p.out = osl ? c->xi : out_inner;
    p.Fi = c->Fi;
    const int sidx = subset < 0 ? g.S : subset;
    p.sens = c->d_sens + (size_t)sidx * g.nx * g.ny;
    p.smax = c->d_smax + sidx;
    p.mask = c->d_mask;
    p.Tp = Tp;
    const int FPT = choose_fpt(Tp);
    p.FG = Tp / FPT;
    p.As = subset < 0 ? g.A : g.A / g.S;
    p.subset = subset;
    p.osl = osl; p.scale = scale; p.beta = beta;
    const int nv = 256 / p.FG;
    p.TX = nv >= 128 ? 32 : (nv >= 64 ? 16 : 8);
    p.TY = nv / p.TX;
    const int nvox = p.TX * p.TY;
    const int threads = nvox * p.FG;
    const int gx = (g.nx + p.TX - 1) / p.TX, gy = (g.ny + p.TY - 1) / p.TY;
    int ZB = 1;
    if (g.nz >= 4 && (long long)gx * gy * ((g.nz + 3) / 4) >= 148LL * 8) ZB = 4;
    else if (g.nz >= 2 && (long long)gx * gy * ((g.nz + 1) / 2) >= 148LL * 8) ZB = 2;
    if (FPT == 12 && ZB == 4) ZB = 2;  // register budget
    dim3 grid(gx, gy, (g.nz + ZB - 1) / ZB);
    const size_t smem = (size_t)KCS_BACK_ACH * nvox * sizeof(float4);
    ProfScope ps(c, KCS_K_BACK);
    switch (FPT) {
        case 4: back_dispatch<4>(ZB, grid, threads, smem, c->stream, g, p); break;
        case 8: back_dispatch<8>(ZB, grid, threads, smem, c->stream, g, p); break;
        default: back_dispatch<12>(ZB, grid, threads, smem, c->stream, g, p); break;
    }
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
    float sum = 0.f;
    for (int la = 0; la < As; ++la) {
        const int a = s == g.S ? la : s + la * g.S;
        const float4 w = voxel_angle_weights(g, a, i, j);
        sum += w.y + w.z + w.w;
    }
    sum *= g.step_mm;
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
__global__ void k_max_nonneg(const float *v, int n, float *out) {
    float m = 0.f;
    for (int q = blockIdx.x * blockDim.x + threadIdx.x; q < n; q += gridDim.x * blockDim.x) m = fmaxf(m, v[q]);
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

int kcs_launch_osl_planar(kcs_ctx *c, float *x, const float *bp, const float *sens, const float *F, float beta,
                          int prior_mode, float sigma2) {
    const KGeom &g = c->g;
    const int v2 = g.nx * g.ny;
    cudaError_t e = cudaMemsetAsync(c->d_tmp_smax, 0, sizeof(float), c->stream);
    if (e != cudaSuccess) { c->err = cudaGetErrorString(e); return KCS_ERR_CUDA; }
    ProfScope ps(c, KCS_K_OTHER);
    k_max_nonneg<<<64, 256, 0, c->stream>>>(sens, v2, c->d_tmp_smax);
    LAUNCH_CHECK(c);
    const size_t n = (size_t)c->cfg.n_frames * c->n_vox;
    k_osl_planar<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(x, bp, sens, F, c->d_mask, c->d_tmp_smax, n, v2, beta,
                                                                     prior_mode, sigma2);
    LAUNCH_CHECK(c);
    return KCS_OK;
}
