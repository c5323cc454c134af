// kcs_static.cu -- kcs_forward_project_static (include/kcs.h): the forward projector for callers that may not allocate
// device memory (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).  No kcs_ctx, no
// cudaMalloc / cudaFree / allocating library routine: the packed volume, the packed sinogram and the angle table that
// kcs_create keeps in its workspace live in ONE file-scope __device__ array of KCS_STATIC_SCRATCH_BYTES, and the kernels
// are the ones kcs_forward_project launches (k_pack, k_forward, k_unpack through their launchers).
//
// The array's name is a host-side stand-in in host code, not a device address: its device address is taken here, in the
// file that defines it, with cudaGetSymbolAddress -- once per device, with that device current -- and handed to the
// kernels as a plain pointer.
#include <climits>
#include <cmath>
#include <mutex>

#include "kcs_internal.cuh"

namespace {

// every GPU on which this entry point has run holds these bytes until the process exits
static __device__ __align__(256) unsigned char g_static_scratch[KCS_STATIC_SCRATCH_BYTES];

constexpr int kMaxDevices = 64;
std::mutex g_mu;
unsigned char *g_scratch_ptr[kMaxDevices] = {};  // device address of g_static_scratch on device d (nullptr: not taken yet)

thread_local std::string g_static_err;

int sfail(int code, const std::string &msg) {
    g_static_err = msg;
    return code;
}

int scratch_of_current_device(unsigned char **out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return sfail(KCS_ERR_CUDA, std::string("kcs_forward_project_static: cudaGetDevice: ") + cudaGetErrorString(e));
    if (dev < 0 || dev >= kMaxDevices) return sfail(KCS_ERR_CUDA, "kcs_forward_project_static: device ordinal beyond 63");
    std::lock_guard<std::mutex> lk(g_mu);
    if (!g_scratch_ptr[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess || !p) {
            cudaGetLastError();
            return sfail(KCS_ERR_CUDA, std::string("kcs_forward_project_static: cudaGetSymbolAddress: ") + cudaGetErrorString(e));
        }
        g_scratch_ptr[dev] = static_cast<unsigned char *>(p);
    }
    *out = g_scratch_ptr[dev];
    return KCS_OK;
}

// a * b, saturating just above the scratch limit (both factors >= 0)
unsigned long long mul_cap(unsigned long long a, unsigned long long b) {
    const unsigned long long cap = (unsigned long long)KCS_STATIC_SCRATCH_BYTES + 1;
    if (a == 0 || b == 0) return 0;
    if (a > cap || b > cap) return cap;
    const unsigned long long p = a * b;  // < 2^52
    return p > cap ? cap : p;
}
unsigned long long round256(unsigned long long n) { return (n + 255ull) & ~255ull; }

// the angle table travels as kernel arguments (copied at launch: no pageable-memory copy, nothing to keep alive)
constexpr int kAngleChunk = 64;
struct AngleChunk {
    double4 v[kAngleChunk];
};
__global__ void k_static_put_angles(AngleChunk ch, int n, double4 *dst) {
    if ((int)threadIdx.x < n) dst[threadIdx.x] = ch.v[threadIdx.x];
}

}  // namespace

extern "C" {

const char *kcs_static_last_error(void) { return g_static_err.c_str(); }

int kcs_forward_project_static(const kcs_config *cfg, const float *x, float *y_s, int subset, int nf, void *stream) {
    if (!cfg || !x || !y_s) return sfail(KCS_ERR_NULL, "kcs_forward_project_static: NULL argument");
    if (cfg->nx <= 0 || cfg->ny <= 0 || cfg->nz <= 0 || cfg->n_angles <= 0 || cfg->n_bins <= 0 || cfg->n_steps <= 0 ||
        cfg->n_subsets <= 0 || !(cfg->vx > 0) || !(cfg->vy > 0) || !(cfg->bin_mm > 0) || !(cfg->step_mm > 0))
        return sfail(KCS_ERR_SHAPE, "kcs_forward_project_static: non-positive size");
    if (cfg->n_angles % cfg->n_subsets != 0) return sfail(KCS_ERR_SUBSET, "kcs_forward_project_static: n_subsets does not divide n_angles");
    if (subset < -1 || subset >= cfg->n_subsets) return sfail(KCS_ERR_SHAPE, "kcs_forward_project_static: subset out of range");
    if (nf <= 0 || nf > KCS_MAX_FRAMES) return sfail(KCS_ERR_FRAMES, "kcs_forward_project_static: nf must be in [1, KCS_MAX_FRAMES]");

    const int nx = cfg->nx, ny = cfg->ny, nz = cfg->nz, A = cfg->n_angles, B = cfg->n_bins;
    const int As = subset < 0 ? A : A / cfg->n_subsets;
    const int Tp = round_up4(nf);
    const int nxp = nx + 2 * KCS_PAD, nyp = ny + 2 * KCS_PAD;
    // scratch: [angle table A double4][xi nz nyp nxp Tp floats][qi nz As B Tp floats], each part on a 256 B boundary
    const unsigned long long b_tab = round256(mul_cap((unsigned long long)A, sizeof(double4)));
    const unsigned long long b_xi = round256(mul_cap(mul_cap(mul_cap((unsigned long long)nz, (unsigned long long)nyp), (unsigned long long)nxp), 4ull * Tp));
    const unsigned long long b_qi = round256(mul_cap(mul_cap(mul_cap((unsigned long long)nz, (unsigned long long)As), (unsigned long long)B), 4ull * Tp));
    const unsigned long long need = b_tab + b_xi + b_qi;
    if (need > (unsigned long long)KCS_STATIC_SCRATCH_BYTES) {
        const bool sat = b_xi > KCS_STATIC_SCRATCH_BYTES || b_qi > KCS_STATIC_SCRATCH_BYTES || b_tab > KCS_STATIC_SCRATCH_BYTES;
        return sfail(KCS_ERR_SHAPE, "kcs_forward_project_static: this geometry needs " + (sat ? std::string("more than ") : std::string()) +
                                        std::to_string(sat ? (unsigned long long)KCS_STATIC_SCRATCH_BYTES : need) +
                                        " bytes of scratch, the static array holds KCS_STATIC_SCRATCH_BYTES = " +
                                        std::to_string((unsigned long long)KCS_STATIC_SCRATCH_BYTES) +
                                        " (use kcs_create + kcs_forward_project for larger problems)");
    }

    unsigned char *scratch = nullptr;
    int rc = scratch_of_current_device(&scratch);
    if (rc != KCS_OK) return rc;
    double4 *d_fwd = reinterpret_cast<double4 *>(scratch);
    float *xi = reinterpret_cast<float *>(scratch + b_tab);
    float *qi = reinterpret_cast<float *>(scratch + b_tab + b_xi);

    // a host-side context that owns nothing: geometry, the three scratch pointers, the caller's stream
    kcs_ctx c{};
    c.stream = (cudaStream_t)stream;
    KGeom &g = c.g;
    g.nx = nx; g.ny = ny; g.nz = nz; g.nzr = nz; g.nxp = nxp; g.nyp = nyp;
    g.A = A; g.B = B; g.K = cfg->n_steps; g.S = cfg->n_subsets;
    g.step_mm = cfg->step_mm; g.bin_mm = cfg->bin_mm;
    g.cx = 0.5 * (nx - 1); g.cy = 0.5 * (ny - 1); g.cb = 0.5 * (B - 1); g.ck = 0.5 * (g.K - 1);
    g.fwd = d_fwd;
    g.bwd = nullptr;  // the forward projector reads g.fwd only
    c.n_vox = (size_t)nz * ny * nx;
    c.n_pix_pad = (size_t)nz * nyp * nxp;
    c.n_ray_all = (size_t)nz * A * B;
    c.xi = xi;
    c.qi = qi;

    // P1: angle table in fp64 on the host, the formula of kcs_create
    for (int a0 = 0; a0 < A; a0 += kAngleChunk) {
        AngleChunk ch;
        const int n = A - a0 < kAngleChunk ? A - a0 : kAngleChunk;
        for (int q = 0; q < n; ++q) {
            const double th = M_PI * (double)(a0 + q) / (double)A, cs = std::cos(th), sn = std::sin(th);
            const double vx = cfg->vx, vy = cfg->vy, bin = cfg->bin_mm, st = cfg->step_mm;
            ch.v[q] = make_double4(bin * cs / vx, -st * sn / vx, bin * sn / vy, st * cs / vy);
        }
        for (int q = n; q < kAngleChunk; ++q) ch.v[q] = make_double4(0.0, 0.0, 0.0, 0.0);
        k_static_put_angles<<<1, kAngleChunk, 0, c.stream>>>(ch, n, d_fwd + a0);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return sfail(KCS_ERR_CUDA, std::string("kcs_forward_project_static: angle table launch: ") + cudaGetErrorString(e));
    }
    // the array keeps the last call's contents: the zero border of the padded volume (P2: outside pixels are 0) and the
    // frames nf..Tp of every pixel must start at 0 -- clear the whole packed volume, every call
    cudaError_t e = cudaMemsetAsync(xi, 0, (size_t)b_xi, c.stream);
    if (e != cudaSuccess) return sfail(KCS_ERR_CUDA, std::string("kcs_forward_project_static: cudaMemsetAsync: ") + cudaGetErrorString(e));
    rc = kcs_launch_pack(&c, x, c.n_vox, nf, xi, Tp, (long long)nz * ny, nx, ny, (long long)nyp * nxp, nxp, KCS_PAD * (nxp + 1));
    if (rc == KCS_OK) rc = kcs_launch_forward(&c, Tp, subset, 0, 1.f, 0, 0, 0, nz);
    if (rc == KCS_OK) rc = kcs_launch_unpack(&c, qi, Tp, y_s, (size_t)nz * As * B, nf, (long long)nz * As, B, INT_MAX, 0, B, 0);
    if (rc != KCS_OK) return sfail(rc, "kcs_forward_project_static: " + c.err);
    return KCS_OK;
}

}  // extern "C"
