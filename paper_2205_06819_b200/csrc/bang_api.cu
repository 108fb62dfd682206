// bang_api.cu -- the C ABI of include/bang.h: context, one-off table kernels, data preparation, launches.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/bang.h"
#include "bang_host.h"
#include "bang_ns.cuh"
#include "bang_slow.cuh"

using namespace bang;

struct bang_ctx {
    bang_grid grid{};
    bang_psf psf{};
    bang_model model{};
    int device = 0;
    cudaStream_t stream = nullptr;
    int n_sm = 0;
    int smem_optin = 0;                    // cudaDevAttrMaxSharedMemoryPerBlockOptin: every kernel is opted in to this maximum
    GridC g{};
    FitC fit{};
    int rk = 0, nacc = 0, P = 0, nxp = 0, threads = 0;
    std::vector<double> W;                 // composite taps, nacc * s
    void* btab = nullptr; int btab_first = 0, btab_cells = 0;
    void* Ftab = nullptr; int Ftab_first = 0, Ftab_cells = 0;
    double2* data = nullptr; double C0 = 0.0; bool has_data = false;
    double* scal = nullptr;                // device scratch: {C0, bad-pixel count}, per-CTA partial sums, the ticket counter
    double* gl_dev = nullptr;              // N_J Gauss-Legendre nodes then weights (reading B): table build, direct path
    double2* qd_dev = nullptr; float2* qf_dev = nullptr;   // the same rule as {a_k, b_k} pairs (reading U', ext_Itilde)
    // staging for the *_host calls
    double* h_theta = nullptr; double* d_theta = nullptr; void* h_out = nullptr; void* d_out = nullptr;
    size_t cap_theta = 0, cap_out = 0;
    long long launches = 0;
    int force_ctas = 0;
    int launch_cache[2] = {0, 0};
    // direct path (bang_slow.cuh): list of the theta k_fused leaves to k_slow, {count, CTAs done}, capacity; 0 = the grid
    // is too large for k_slow's shared memory (such theta are then reported as out of domain)
    int* slow_list = nullptr; int* slow_cnt = nullptr; int slow_cap = 0; size_t slow_smem = 0;
    int* na_scratch = nullptr;             // device address of g_noalloc_scratch on this context's device (bang_loglike_noalloc)
    double* W_dev = nullptr;               // composite taps on the device (direct path)
    bool fine_ready = false;               // k_fine's shared-memory opt-in done (once per context)
    // bang_ns_walk scratch: proposals [K][d], their theta [K][17] and likelihoods [K], Cholesky factors + scales, counts
    double* ns_prop = nullptr; double* ns_theta = nullptr; double* ns_pl = nullptr; double* ns_chol = nullptr;
    int* ns_acc = nullptr; int ns_capK = 0, ns_capG = 0;
    char err[512] = {0};
};

// ---- scratch of the allocation-free entry point (bang_loglike_noalloc) ---------------------------------------------------
// The fused kernel hands the theta whose radii leave its tables to the direct-path kernel through a list in device memory
// (bang_slow.cuh); bang_loglike keeps that list in a cudaMalloc'ed buffer that grows with B.  Callers that must not
// allocate (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc) get the same two kernels with the list in
// this file-scope array instead: [0] = number of entries, [1] = CTAs of k_slow that have finished, [64 ..] = the entries.
// 256 KiB + 256 B, held by every GPU that loads the library until the process exits.  ONE array per device, shared by every
// call and every context: calls that overlap on the GPU (two streams) race on it.
#define BANG_NOALLOC_MAX_B_IMPL 65536
static __device__ __align__(256) int g_noalloc_scratch[64 + BANG_NOALLOC_MAX_B_IMPL];
static_assert(BANG_NOALLOC_MAX_B_IMPL == BANG_NOALLOC_MAX_B, "include/bang.h states the limit");
// In host code `g_noalloc_scratch` is a host-side stand-in for the symbol, NOT a device address: the address a kernel may be
// given comes from cudaGetSymbolAddress, asked once per device with that device current (bang_create).
constexpr int kMaxDevices = 64;
static int* g_noalloc_ptr[kMaxDevices] = {nullptr};

namespace {

// device address of the scratch array on the CURRENT device (which must be `device`); NULL + the CUDA error on failure
cudaError_t noalloc_scratch_address(int device, int** out) {
    *out = nullptr;
    if (device < 0 || device >= kMaxDevices) return cudaErrorInvalidDevice;
    if (!g_noalloc_ptr[device]) {
        int* ptr = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void**)&ptr, g_noalloc_scratch);
        if (e != cudaSuccess) return e;
        g_noalloc_ptr[device] = ptr;
    }
    *out = g_noalloc_ptr[device];
    return cudaSuccess;
}

int fail(bang_ctx* c, int code, const char* fmt, ...) {
    if (c) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(c->err, sizeof(c->err), fmt, ap);
        va_end(ap);
    }
    return code;
}
#define CU(call)                                                                                              \
    do {                                                                                                      \
        cudaError_t e_ = (call);                                                                              \
        if (e_ != cudaSuccess)                                                                                \
            return fail(ctx, e_ == cudaErrorMemoryAllocation ? BANG_ENOMEM : BANG_ECUDA, "%s: %s", #call,    \
                        cudaGetErrorString(e_));                                                              \
    } while (0)

// Every entry point runs on the context's device and leaves the calling thread's current device as it found it.
struct DeviceGuard {
    int prev = -1;
    bool ok = false;
    explicit DeviceGuard(int dev) {
        if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
        ok = (prev == dev) || cudaSetDevice(dev) == cudaSuccess;
        if (prev == dev) prev = -1;                    // nothing to restore
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
    DeviceGuard(const DeviceGuard&) = delete;
    DeviceGuard& operator=(const DeviceGuard&) = delete;
};
#define ON_DEVICE(ctx)                                                                       \
    DeviceGuard dev_guard_((ctx)->device);                                                   \
    if (!dev_guard_.ok) return fail((ctx), BANG_ECUDA, "cudaSetDevice(%d) failed", (ctx)->device)

// Gauss-Legendre nodes and weights on (-1,1): Newton iteration on P_n (Abramowitz & Stegun 25.4.29), long double
void gauss_legendre(int n, double* x, double* w) {
    for (int i = 0; i < (n + 1) / 2; ++i) {
        long double z = cosl(3.14159265358979323846264338328L * (i + 0.75L) / (n + 0.5L)), pp = 1;
        for (int it = 0; it < 100; ++it) {
            long double p0 = 1, p1 = z;
            for (int j = 2; j <= n; ++j) {
                long double p2 = ((2 * j - 1) * z * p1 - (j - 1) * p0) / j;
                p0 = p1; p1 = p2;
            }
            pp = n * (z * p1 - p0) / (z * z - 1);
            long double dz = p1 / pp;
            z -= dz;
            if (fabsl(dz) < 1e-19L) break;
        }
        {   // derivative at the converged root
            long double p0 = 1, p1 = z;
            for (int j = 2; j <= n; ++j) {
                long double p2 = ((2 * j - 1) * z * p1 - (j - 1) * p0) / j;
                p0 = p1; p1 = p2;
            }
            pp = n * (z * p1 - p0) / (z * z - 1);
        }
        x[i] = (double)-z; x[n - 1 - i] = (double)z;
        w[i] = w[n - 1 - i] = (double)(2 / ((1 - z * z) * pp * pp));
    }
}

// Chebyshev nodes t_k = cos(pi (k + 1/2)/(D+1)) and the inverse of the Vandermonde matrix V[k][d] = t_k^d
void make_fit(int D, FitC& fit) {
    const int n = D + 1;
    long double A[8][16];
    for (int k = 0; k < n; ++k) {
        long double t = cosl(3.14159265358979323846264338328L * (k + 0.5L) / n), p = 1;
        fit.tnode[k] = (double)t;
        for (int d = 0; d < n; ++d) { A[k][d] = p; p *= t; }
        for (int d = 0; d < n; ++d) A[k][n + d] = (d == k) ? 1 : 0;
    }
    for (int c = 0; c < n; ++c) {                      // Gauss-Jordan with partial pivoting
        int piv = c;
        for (int r = c + 1; r < n; ++r) if (fabsl(A[r][c]) > fabsl(A[piv][c])) piv = r;
        for (int j = 0; j < 2 * n; ++j) { long double t = A[c][j]; A[c][j] = A[piv][j]; A[piv][j] = t; }
        long double inv = 1 / A[c][c];
        for (int j = 0; j < 2 * n; ++j) A[c][j] *= inv;
        for (int r = 0; r < n; ++r)
            if (r != c) {
                long double f = A[r][c];
                for (int j = 0; j < 2 * n; ++j) A[r][j] -= f * A[c][j];
            }
    }
    for (int d = 0; d < n; ++d)
        for (int k = 0; k < n; ++k) fit.vinv[d * n + k] = (double)A[d][n + k];
}

// ---- one-off kernels: the scale-free tables (K0) ---------------------------------------------
// which = 0: the bulge's SigmaTilde(s) and N_J-node Jeans integral J(s) (Hernquist or Jaffe), at u = s^2;
// which = 1: Freeman F(y), u = y^2
template <typename T>
__global__ void k_univ_nodes(int which, int bulge_profile, int first, int n_cells, FitC fit, int NJ,
                             const double* __restrict__ glx, const double* __restrict__ glw, double* __restrict__ vals) {
    constexpr int NC = TabCfg<T>::D + 1;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_cells * NC) return;
    const int cell = i / NC, k = i - cell * NC;
    double lo, width;
    tab_interval<T>(first + cell, lo, width);
    const double x = sqrt(lo + 0.5 * width * (fit.tnode[k] + 1.0));
    if (which == 0) {
        vals[(cell * 2 + 0) * NC + k] = bulge_profile == 1 ? jaffe_sigma_tilde(x) : sigma_tilde(x);
        vals[(cell * 2 + 1) * NC + k] = bulge_profile == 1 ? jaffe_jeans_J(x, NJ, glx, glw) : jeans_J(x, NJ, glx, glw);
    } else {
        vals[cell * NC + k] = freeman_F(x);
    }
}
template <typename T>
__global__ void k_univ_fit(int n_rows, FitC fit, const double* __restrict__ vals, T* __restrict__ coef) {
    constexpr int NC = TabCfg<T>::D + 1;
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n_rows) return;
    for (int d = 0; d < NC; ++d) {
        double a = 0.0;
        for (int k = 0; k < NC; ++k) a = fma(fit.vinv[d * NC + k], vals[r * NC + k], a);
        coef[r * NC + d] = (T)a;
    }
}

// data preparation (layout [ny][4][P][gmax], gmax >= nxp/P the pixel-group pitch of the launch's thread class; the
// caller zeroes the buffer): {d, 1/e} per used pixel ({0,0} where masked or padded), C0 = sum -1/2 ln(2 pi e^2), and the number
// of used pixels with err <= 0 or a non-finite value.  A grid of CTAs; per-CTA partial sums go to scal[2 + 2 blk ..] and the
// last CTA to finish adds them in CTA order: the reduction order is fixed, the result deterministic.
constexpr int kPrepMaxBlocks = 64;
__global__ void __launch_bounds__(256) k_prep_data(int nx, int ny, int nxp, int P, int gmax, const double* __restrict__ data,
                                                   const double* __restrict__ err, const unsigned char* __restrict__ mask,
                                                   double2* __restrict__ out, double* __restrict__ scal, unsigned* __restrict__ ticket) {
    __shared__ double sh[2][8];
    __shared__ bool last;
    double c0 = 0.0, bad = 0.0;
    const int total = ny * 4 * nxp;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < total; i += gridDim.x * blockDim.x) {
        const int px = i % nxp, q = (i / nxp) % 4, py = i / (4 * nxp);
        double2 v = make_double2(0.0, 0.0);
        if (px < nx) {
            const size_t src = ((size_t)q * ny + py) * nx + px;
            if (mask[src]) {
                const double d = data[src], e = err[src];
                if (!(e > 0.0) || !isfinite(e) || !isfinite(d)) bad += 1.0;
                else {
                    v = make_double2(d, 1.0 / e);
                    c0 += -0.5 * log(2.0 * kPi * e * e);
                }
            }
        }
        // [py][q][i][group]: pixel px = group P + i, so that the fused kernel's load of its i-th pixel is coalesced
        out[(((size_t)py * 4 + q) * P + px % P) * gmax + px / P] = v;
    }
    for (int o = 16; o > 0; o >>= 1) {
        c0 += __shfl_xor_sync(0xffffffffu, c0, o);
        bad += __shfl_xor_sync(0xffffffffu, bad, o);
    }
    if ((threadIdx.x & 31) == 0) { sh[0][threadIdx.x >> 5] = c0; sh[1][threadIdx.x >> 5] = bad; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double a = 0.0, b = 0.0;
        for (int w = 0; w < (int)(blockDim.x + 31) / 32; ++w) { a += sh[0][w]; b += sh[1][w]; }
        scal[2 + 2 * blockIdx.x] = a; scal[3 + 2 * blockIdx.x] = b;
        __threadfence();
        last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (last && threadIdx.x == 0) {
        __threadfence();
        double a = 0.0, b = 0.0;
        for (unsigned k = 0; k < gridDim.x; ++k) { a += scal[2 + 2 * k]; b += scal[3 + 2 * k]; }
        scal[0] = a; scal[1] = b;
        *ticket = 0u;
    }
}

// ---- peak probes (bang_probe_peaks): 8 independent chains per thread, no memory traffic --------------------------------
template <int WHICH>
__global__ void __launch_bounds__(256) k_probe(int iters, float seed, float* __restrict__ sink) {
    float a[8];
    double d[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) { a[i] = seed + (float)(threadIdx.x + i) * 1e-3f; d[i] = (double)a[i]; }
    const float m = 0.999f + seed * 1e-6f, c = 1e-3f;
    const double md = (double)m, cd = (double)c;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                if (WHICH == 0) a[i] = fmaf(a[i], m, c);
                else if (WHICH == 1) a[i] = fast_exp2(a[i]) - 1.0f;          // one MUFU.EX2 + one FADD per step
                else d[i] = fma(d[i], md, cd);
            }
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += a[i] + (float)d[i];
    if (s == 12345.678f) sink[0] = s;                                     // keeps the chains alive, never true in practice
}

// eq. 20 + App. C error model (bang_ml_from_colour): elementwise, HBM-bound (48 B per pixel), grid-stride
__global__ void k_ml_from_colour(const double* __restrict__ mb, const double* __restrict__ mg, const double* __restrict__ dmb,
                                 const double* __restrict__ dmg, long long n, double a, double b, double sig,
                                 double* __restrict__ ml, double* __restrict__ mlerr) {
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const double logml = fma(b, mb[i] - mg[i], a);
        const double dlog = sqrt(fma(b * b, fma(dmb[i], dmb[i], dmg[i] * dmg[i]), sig * sig));
        const double v = exp10(logml);
        ml[i] = v;
        mlerr[i] = 2.302585092994045684 * v * dlog;
    }
}

template <typename T>
int build_universal(bang_ctx* ctx, const double* glx_dev, const double* glw_dev) {
    constexpr int NC = TabCfg<T>::D + 1;
    ctx->btab_first = tab_first_cell<T>(kBulgeOctLo);
    ctx->btab_cells = (kBulgeOctHi - kBulgeOctLo) << TabCfg<T>::M;
    ctx->Ftab_first = tab_first_cell<T>(kFOctLo);
    ctx->Ftab_cells = (kFOctHi - kFOctLo) << TabCfg<T>::M;
    double* vals = nullptr;
    const size_t nb = (size_t)ctx->btab_cells * 2 * NC, nf = (size_t)ctx->Ftab_cells * NC;
    CU(cudaMalloc(&vals, (nb + nf) * sizeof(double)));
    struct Free { double* p; ~Free() { cudaFree(p); } } free_vals{vals};      // also on the error returns below
    CU(cudaMalloc(&ctx->btab, nb * sizeof(T)));
    CU(cudaMalloc(&ctx->Ftab, nf * sizeof(T)));
    const int th = 128;
    k_univ_nodes<T><<<(ctx->btab_cells * NC + th - 1) / th, th, 0, ctx->stream>>>(0, ctx->model.bulge_profile, ctx->btab_first, ctx->btab_cells, ctx->fit,
                                                                                ctx->model.jeans_nodes, glx_dev, glw_dev, vals);
    k_univ_nodes<T><<<(ctx->Ftab_cells * NC + th - 1) / th, th, 0, ctx->stream>>>(1, 0, ctx->Ftab_first, ctx->Ftab_cells, ctx->fit, 0,
                                                                                nullptr, nullptr, vals + nb);
    k_univ_fit<T><<<(ctx->btab_cells * 2 + th - 1) / th, th, 0, ctx->stream>>>(ctx->btab_cells * 2, ctx->fit, vals,
                                                                             static_cast<T*>(ctx->btab));
    k_univ_fit<T><<<(ctx->Ftab_cells + th - 1) / th, th, 0, ctx->stream>>>(ctx->Ftab_cells, ctx->fit, vals + nb,
                                                                         static_cast<T*>(ctx->Ftab));
    ctx->launches += 4;
    CU(cudaGetLastError());
    CU(cudaStreamSynchronize(ctx->stream));
    return BANG_OK;
}

cudaError_t dispatch_fused(const bang_ctx* c, const FusedLaunch& L, FusedInfo* info, bool query) {
    const bool f64 = c->model.precision == BANG_FP64;
    switch (c->g.s) {
        case 1: return f64 ? launch_fused_double_1(L, info, query) : launch_fused_float_1(L, info, query);
        case 2: return f64 ? launch_fused_double_2(L, info, query) : launch_fused_float_2(L, info, query);
        case 3: return f64 ? launch_fused_double_3(L, info, query) : launch_fused_float_3(L, info, query);
        case 4: return f64 ? launch_fused_double_4(L, info, query) : launch_fused_float_4(L, info, query);
        default: return cudaErrorInvalidValue;
    }
}

QuadC make_quad(const bang_ctx* c) {
    QuadC q{};
    q.qd = c->qd_dev; q.qf = c->qf_dev; q.NJ = c->model.jeans_nodes;
    // coarse panels of the per-theta Itilde_ext build (bang_kernels.cuh): 8 nodes per 2 octaves in fp32 mode, 12 per octave in fp64
    q.ND = c->model.precision == BANG_FP64 ? 12 : 8;
    q.span = c->model.precision == BANG_FP64 ? 1 : 2;
    for (int k = 0; k < q.ND; ++k) {
        const long double a = 3.14159265358979323846264338328L * (2 * k + 1) / (2.0L * q.ND);
        q.bx[k] = (double)cosl(a);
        q.bw[k] = (double)((k & 1 ? -1.0L : 1.0L) * sinl(a));
    }
    return q;
}
DirectC make_direct(const bang_ctx* c) {
    return DirectC{c->gl_dev, c->gl_dev + c->model.jeans_nodes, c->model.jeans_nodes, make_quad(c)};
}

FusedLaunch make_launch(bang_ctx* c, const double* theta, int B, int mode, void* maps, double* logL) {
    FusedLaunch L{};
    L.g = c->g; L.fit = c->fit;
    L.btab = c->btab; L.btab_first = c->btab_first; L.btab_cells = c->btab_cells;
    L.Ftab = c->Ftab; L.Ftab_first = c->Ftab_first; L.Ftab_cells = c->Ftab_cells;
    L.quad = make_quad(c);
    L.W = c->W.data(); L.nacc = c->nacc;
    L.theta = theta; L.B = B; L.P = c->P; L.nxp = c->nxp; L.mode = mode;
    L.maps = maps; L.data = c->data; L.C0 = c->C0; L.logL = logL;
    L.threads = c->threads; L.ctas = c->force_ctas; L.n_sm = c->n_sm; L.smem_optin = c->smem_optin; L.stream = c->stream;
    L.cache = c->launch_cache;
    L.slow_list = c->slow_smem ? c->slow_list : nullptr; L.slow_count = c->slow_cnt;
    return L;
}

// pitch of the data array's pixel-group axis: the launch-bound class of the fused kernel / 4 (lbc_threads)
int data_gmax(const bang_ctx* c) { return (c->threads <= 128 ? 128 : (c->threads <= 256 ? 256 : 512)) / 4; }

// room for B entries in the list of theta that take the direct path
int ensure_slow_list(bang_ctx* ctx, int B) {
    if (!ctx->slow_smem || B <= ctx->slow_cap) return BANG_OK;
    CU(cudaStreamSynchronize(ctx->stream));
    cudaFree(ctx->slow_list); ctx->slow_list = nullptr; ctx->slow_cap = 0;
    CU(cudaMalloc(&ctx->slow_list, (size_t)B * sizeof(int)));
    ctx->slow_cap = B;
    return BANG_OK;
}

// the direct path for the theta k_fused recorded (an empty list costs one empty launch)
template <typename T>
int run_slow(bang_ctx* ctx, const double* theta_dev, int mode, void* maps_dev, double* logL_dev) {
    if (!ctx->slow_smem) return BANG_OK;
    SlowParams<T> p{};
    p.g = ctx->g;
    p.btab = PolyTab<T>{static_cast<const T*>(ctx->btab), ctx->btab_first, ctx->btab_cells};
    p.Ftab = PolyTab<T>{static_cast<const T*>(ctx->Ftab), ctx->Ftab_first, ctx->Ftab_cells};
    p.direct = make_direct(ctx);
    p.W = ctx->W_dev; p.nacc = ctx->nacc;
    p.theta = theta_dev; p.slow_list = ctx->slow_list; p.slow_count = ctx->slow_cnt; p.done = ctx->slow_cnt + 1;
    p.maps = static_cast<T*>(maps_dev); p.data = ctx->data; p.P = ctx->P; p.gmax = data_gmax(ctx);
    p.C0 = ctx->C0; p.logL = logL_dev;
    if (mode == 0) k_slow<T, 0><<<ctx->n_sm, 256, ctx->slow_smem, ctx->stream>>>(p);
    else k_slow<T, 1><<<ctx->n_sm, 256, ctx->slow_smem, ctx->stream>>>(p);
    ctx->launches += 1;
    CU(cudaGetLastError());
    return BANG_OK;
}
// bang_loglike with no allocation anywhere on its path: the same k_fused + k_slow launches, the direct-path list in the
// file-scope array above.  No cudaMalloc / cudaFree / allocating routine is called here or below (make_launch, the launchers
// and fail() use fixed storage; the first call per context does the kernel's shared-memory opt-in and occupancy query).
template <typename T>
int run_slow_noalloc(bang_ctx* ctx, const double* theta_dev, double* logL_dev) {
    if (!ctx->slow_smem) return BANG_OK;
    SlowParams<T> p{};
    p.g = ctx->g;
    p.btab = PolyTab<T>{static_cast<const T*>(ctx->btab), ctx->btab_first, ctx->btab_cells};
    p.Ftab = PolyTab<T>{static_cast<const T*>(ctx->Ftab), ctx->Ftab_first, ctx->Ftab_cells};
    p.direct = make_direct(ctx);
    p.W = ctx->W_dev; p.nacc = ctx->nacc;
    p.theta = theta_dev; p.slow_list = ctx->na_scratch + 64; p.slow_count = ctx->na_scratch; p.done = ctx->na_scratch + 1;
    p.maps = nullptr; p.data = ctx->data; p.P = ctx->P; p.gmax = data_gmax(ctx);
    p.C0 = ctx->C0; p.logL = logL_dev;
    k_slow<T, 1><<<ctx->n_sm, 256, ctx->slow_smem, ctx->stream>>>(p);
    ctx->launches += 1;
    CU(cudaGetLastError());
    return BANG_OK;
}

template <typename T>
int setup_slow(bang_ctx* ctx) {
    const size_t smem = slow_smem_bytes<T>(ctx->g, ctx->nacc);
    cudaDeviceProp prop;
    CU(cudaGetDeviceProperties(&prop, ctx->device));
    if (smem > prop.sharedMemPerBlockOptin) return BANG_OK;          // slow_smem stays 0: no direct path on this grid
    // opted in to the device maximum, not to this context's size: the attribute is per function, and another context
    // of the same instantiation may need more
    CU(cudaFuncSetAttribute(k_slow<T, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)prop.sharedMemPerBlockOptin));
    CU(cudaFuncSetAttribute(k_slow<T, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)prop.sharedMemPerBlockOptin));
    CU(cudaMalloc(&ctx->slow_cnt, 2 * sizeof(int)));
    CU(cudaMemsetAsync(ctx->slow_cnt, 0, 2 * sizeof(int), ctx->stream));
    ctx->slow_smem = smem;
    return BANG_OK;
}

int ensure_staging(bang_ctx* ctx, int B, size_t out_bytes) {
    const size_t tb = (size_t)B * kNTheta * sizeof(double);
    if (tb > ctx->cap_theta) {
        if (ctx->h_theta) cudaFreeHost(ctx->h_theta);
        if (ctx->d_theta) cudaFree(ctx->d_theta);
        ctx->h_theta = nullptr; ctx->d_theta = nullptr; ctx->cap_theta = 0;
        CU(cudaMallocHost(&ctx->h_theta, tb));
        CU(cudaMalloc(&ctx->d_theta, tb));
        ctx->cap_theta = tb;
    }
    if (out_bytes > ctx->cap_out) {
        if (ctx->h_out) cudaFreeHost(ctx->h_out);
        if (ctx->d_out) cudaFree(ctx->d_out);
        ctx->h_out = nullptr; ctx->d_out = nullptr; ctx->cap_out = 0;
        CU(cudaMallocHost(&ctx->h_out, out_bytes));
        CU(cudaMalloc(&ctx->d_out, out_bytes));
        ctx->cap_out = out_bytes;
    }
    return BANG_OK;
}

}  // namespace

extern "C" {

const char* bang_strerror(int code) {
    switch (code) {
        case BANG_OK: return "success";
        case BANG_EINVAL: return "invalid argument or unsupported configuration";
        case BANG_ENOMEM: return "out of memory";
        case BANG_ECUDA: return "CUDA error";
        case BANG_ENODATA: return "no data loaded (call bang_set_data first)";
        default: return "unknown error";
    }
}

const char* bang_last_error(const bang_ctx* ctx) { return ctx ? ctx->err : ""; }

long long bang_launch_count(const bang_ctx* ctx) { return ctx ? ctx->launches : 0; }

int bang_get_geometry(const bang_ctx* ctx, int* r_k, int* nfx, int* nfy) {
    if (!ctx) return BANG_EINVAL;
    if (r_k) *r_k = ctx->rk;
    if (nfx) *nfx = ctx->g.nfx;
    if (nfy) *nfy = ctx->g.nfy;
    return BANG_OK;
}

int bang_ml_from_colour(const double* m_beta_dev, const double* m_gamma_dev, const double* dm_beta_dev,
                        const double* dm_gamma_dev, long long n, double a, double b, double sigma_alpha, double* ml_dev,
                        double* ml_err_dev, int device, void* cuda_stream) {
    if (n < 0 || (n > 0 && (!m_beta_dev || !m_gamma_dev || !dm_beta_dev || !dm_gamma_dev || !ml_dev || !ml_err_dev))) return BANG_EINVAL;
    if (n == 0) return BANG_OK;
    DeviceGuard dg(device);
    if (!dg.ok) return BANG_ECUDA;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return BANG_ECUDA;
    const int threads = 256;
    const long long want = (n + threads - 1) / threads;
    const int grid = (int)std::min<long long>(want, (long long)prop.multiProcessorCount * 8);
    k_ml_from_colour<<<grid, threads, 0, static_cast<cudaStream_t>(cuda_stream)>>>(m_beta_dev, m_gamma_dev, dm_beta_dev, dm_gamma_dev,
                                                                                  n, a, b, sigma_alpha, ml_dev, ml_err_dev);
    return cudaGetLastError() == cudaSuccess ? BANG_OK : BANG_ECUDA;
}

int bang_probe_peaks(bang_ctx* ctx, double* out_host) {
    if (!ctx) return BANG_EINVAL;
    if (!out_host) return fail(ctx, BANG_EINVAL, "bang_probe_peaks: null pointer");
    ON_DEVICE(ctx);
    float* sink = nullptr;
    CU(cudaMalloc(&sink, sizeof(float)));
    cudaEvent_t e0, e1;
    CU(cudaEventCreate(&e0)); CU(cudaEventCreate(&e1));
    const int grid = ctx->n_sm * 8, threads = 256, iters = 4096;
    for (int which = 0; which < 3; ++which) {
        const int it = which == 0 ? iters : iters / 4;
        float best = 1e30f;
        for (int rep = 0; rep < 4; ++rep) {                                 // first repetition warms up
            cudaEventRecord(e0, ctx->stream);
            if (which == 0) k_probe<0><<<grid, threads, 0, ctx->stream>>>(it, 0.5f, sink);
            else if (which == 1) k_probe<1><<<grid, threads, 0, ctx->stream>>>(it, 0.5f, sink);
            else k_probe<2><<<grid, threads, 0, ctx->stream>>>(it, 0.5f, sink);
            cudaEventRecord(e1, ctx->stream);
            cudaError_t e = cudaEventSynchronize(e1);
            if (e != cudaSuccess) { cudaFree(sink); return fail(ctx, BANG_ECUDA, "bang_probe_peaks: %s", cudaGetErrorString(e)); }
            float ms = 0.f;
            cudaEventElapsedTime(&ms, e0, e1);
            if (rep > 0 && ms < best) best = ms;
            ctx->launches += 1;
        }
        out_host[which] = (double)grid * threads * (double)it * 32.0 / (best * 1e-3);   // 4 x 8 chain steps per iteration
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(sink);
    return BANG_OK;
}

void bang_destroy(bang_ctx* ctx) {
    if (!ctx) return;
    DeviceGuard dg(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    cudaFree(ctx->btab); cudaFree(ctx->Ftab); cudaFree(ctx->data); cudaFree(ctx->scal); cudaFree(ctx->gl_dev); cudaFree(ctx->qd_dev); cudaFree(ctx->qf_dev);
    cudaFree(ctx->d_theta); cudaFree(ctx->d_out);
    cudaFree(ctx->slow_list); cudaFree(ctx->slow_cnt);
    cudaFree(ctx->W_dev);
    cudaFree(ctx->ns_prop); cudaFree(ctx->ns_theta); cudaFree(ctx->ns_pl); cudaFree(ctx->ns_chol); cudaFree(ctx->ns_acc);
    if (ctx->h_theta) cudaFreeHost(ctx->h_theta);
    if (ctx->h_out) cudaFreeHost(ctx->h_out);
    delete ctx;
}

int bang_create(bang_ctx** out, const bang_grid* grid, const bang_psf* psf, const bang_model* model, int device,
                void* cuda_stream) {
    if (!out) return BANG_EINVAL;
    *out = nullptr;
    if (!grid || !psf || !model) return BANG_EINVAL;
    if (grid->nx < 1 || grid->ny < 1 || grid->supersample < 1 || grid->supersample > 4 || !(grid->pix_arcsec > 0) ||
        !(grid->dist_mpc > 0) || !std::isfinite(grid->pix_arcsec) || !std::isfinite(grid->dist_mpc))
        return BANG_EINVAL;
    if (!(psf->sigma_pix >= 0) || !(psf->trunc_nsigma >= 0) || !std::isfinite(psf->sigma_pix) || !std::isfinite(psf->trunc_nsigma))
        return BANG_EINVAL;
    if (!(model->components & (BANG_BULGE | BANG_DISC1 | BANG_DISC2)) || (model->components & ~15u)) return BANG_EINVAL;
    if (model->bulge_profile != BANG_BULGE_HERNQUIST && model->bulge_profile != BANG_BULGE_JAFFE) return BANG_EINVAL;
    if (model->halo_profile != BANG_HALO_HERNQUIST && model->halo_profile != BANG_HALO_NFW) return BANG_EINVAL;
    if (model->jeans_nodes < 1 || model->jeans_nodes > 4096) return BANG_EINVAL;
    if (model->precision != BANG_FP32 && model->precision != BANG_FP64) return BANG_EINVAL;
    if (model->psf_weighting != BANG_PSF_FIELDS && model->psf_weighting != BANG_PSF_FLUX) return BANG_EINVAL;
    if (model->bulge_potential != BANG_POTENTIAL_SELF && model->bulge_potential != BANG_POTENTIAL_TOTAL) return BANG_EINVAL;

    const int s = grid->supersample;
    const int rk = (int)std::ceil(psf->trunc_nsigma * psf->sigma_pix * s - 1e-9);
    const int nacc = round_nacc((2 * rk + s + s - 1) / s);
    if (nacc < 0) return BANG_EINVAL;

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) return BANG_ECUDA;
    DeviceGuard dg(device);
    if (!dg.ok) return BANG_ECUDA;

    bang_ctx* ctx = new (std::nothrow) bang_ctx;
    if (!ctx) return BANG_ENOMEM;
    ctx->grid = *grid; ctx->psf = *psf; ctx->model = *model; ctx->device = device;
    ctx->stream = static_cast<cudaStream_t>(cuda_stream);
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) { delete ctx; return BANG_ECUDA; }
    ctx->n_sm = prop.multiProcessorCount;
    ctx->smem_optin = (int)prop.sharedMemPerBlockOptin;

    const bool f64 = model->precision == BANG_FP64;
    ctx->rk = rk; ctx->nacc = nacc;
    GridC& g = ctx->g;
    g.nx = grid->nx; g.ny = grid->ny; g.s = s; g.rk = rk;
    g.nfx = grid->nx * s + 2 * rk; g.nfy = grid->ny * s + 2 * rk;
    g.jsx = rk - 0.5 + 0.5 * grid->nx * s; g.jsy = rk - 0.5 + 0.5 * grid->ny * s;
    g.spx = s / grid->pix_arcsec;
    g.h = grid->pix_arcsec * grid->dist_mpc * kKpcPerArcsecPerMpc / s;
    g.comps = model->components; g.halo_profile = model->halo_profile; g.bulge_profile = model->bulge_profile;
    g.flux = model->psf_weighting;
    g.bulge_potential = model->bulge_potential;

    // eq. 21 on the fine grid, separable (reading F): g[m] = exp(-m^2/(2 sigma_f^2)), normalised;
    // composed with the s-cell box of the rebin: W[t] = (1/s) sum_{b<s} g[t - b], t = 0 .. 2 r_k + s - 1.
    {
        std::vector<long double> gk(2 * rk + 1);
        const long double sf = (long double)psf->sigma_pix * s;
        long double sum = 0;
        for (int m = -rk; m <= rk; ++m) {
            gk[m + rk] = sf > 0 ? expl(-0.5L * m * m / (sf * sf)) : (m == 0 ? 1.0L : 0.0L);
            sum += gk[m + rk];
        }
        ctx->W.assign((size_t)nacc * s, 0.0);
        for (int t = 0; t < 2 * rk + s; ++t) {
            long double a = 0;
            for (int b = 0; b < s; ++b) {
                const int m = t - b;
                if (m >= 0 && m <= 2 * rk) a += gk[m];
            }
            ctx->W[t] = (double)(a / sum / s);
        }
    }

    // launch shape: P data pixels per thread in the PSF phase, one thread per (observable, pixel group)
    int P = f64 ? 2 : 4;      // fp32: four pixels per PSF thread (the window is read 2.5 times over instead of 4)
#ifdef BANG_TUNING      // development builds only (-DBANG_TUNING): sweep the launch shape from the environment
    if (const char* e = getenv("BANG_P")) if (!f64 && (atoi(e) == 2 || atoi(e) == 4)) P = atoi(e);
#endif
    ctx->P = P;
    ctx->nxp = (grid->nx + P - 1) / P * P;
    const int items = 4 * ctx->nxp / P;
    ctx->threads = std::max(128, (items + 31) / 32 * 32);
    // fp32 maps of up to 64 columns: 64-thread CTAs, all of them PSF threads at P = 4; seven are resident per SM (shared
    // memory), so a batch of 1024 still runs in one round (measured against P = 2 with 128 threads: 0.2336 / 0.2364 ms at
    // B = 1024, 1.730 / 1.778 ms at B = 8192 on the 64 x 64 map)
    if (!f64 && P == 4 && items <= 64) ctx->threads = 64;
#ifdef BANG_TUNING
    if (const char* e = getenv("BANG_THREADS")) if (atoi(e) >= (items + 31) / 32 * 32 && atoi(e) <= 512) ctx->threads = atoi(e) / 32 * 32;
    if (const char* e = getenv("BANG_CTAS")) if (atoi(e) > 0) ctx->force_ctas = atoi(e);
#endif
    if (ctx->threads > 512) { delete ctx; return BANG_EINVAL; }      // row too wide for one CTA
    make_fit(f64 ? TabCfg<double>::D : TabCfg<float>::D, ctx->fit);

    // N_J-node Gauss-Legendre rule (reading B), then the scale-free tables on the device
    std::vector<double> gl(2 * (size_t)model->jeans_nodes);
    gauss_legendre(model->jeans_nodes, gl.data(), gl.data() + model->jeans_nodes);
    int rc = BANG_OK;
    do {
        if (cudaMalloc(&ctx->gl_dev, gl.size() * sizeof(double)) != cudaSuccess) { rc = BANG_ENOMEM; break; }
        if (cudaMemcpyAsync(ctx->gl_dev, gl.data(), gl.size() * sizeof(double), cudaMemcpyHostToDevice, ctx->stream) != cudaSuccess) {
            rc = BANG_ECUDA; break;
        }
        {   // the rule in the form ext_Itilde takes (reading U'): a_k = t^2/(1-t), b_k = w t (2-t)/(1-t)^2 on t in (0,1)
            const int NJ = model->jeans_nodes;
            std::vector<double2> qd(NJ);
            std::vector<float2> qf(NJ);
            for (int k = 0; k < NJ; ++k) {
                const long double t = 0.5L * ((long double)gl[k] + 1.0L), w = 0.5L * (long double)gl[NJ + k];
                const long double a = t * t / (1.0L - t), b = w * t * (2.0L - t) / ((1.0L - t) * (1.0L - t));
                qd[k] = make_double2((double)a, (double)b);
                qf[k] = make_float2((float)a, (float)b);
            }
            if (cudaMalloc(&ctx->qd_dev, NJ * sizeof(double2)) != cudaSuccess || cudaMalloc(&ctx->qf_dev, NJ * sizeof(float2)) != cudaSuccess) {
                rc = BANG_ENOMEM; break;
            }
            if (cudaMemcpy(ctx->qd_dev, qd.data(), NJ * sizeof(double2), cudaMemcpyHostToDevice) != cudaSuccess ||
                cudaMemcpy(ctx->qf_dev, qf.data(), NJ * sizeof(float2), cudaMemcpyHostToDevice) != cudaSuccess) { rc = BANG_ECUDA; break; }
        }
        rc = f64 ? build_universal<double>(ctx, ctx->gl_dev, ctx->gl_dev + model->jeans_nodes)
                 : build_universal<float>(ctx, ctx->gl_dev, ctx->gl_dev + model->jeans_nodes);
        if (rc != BANG_OK) break;
        if (cudaMalloc(&ctx->scal, (4 + 2 * kPrepMaxBlocks) * sizeof(double)) != cudaSuccess) { rc = BANG_ENOMEM; break; }
        if (cudaMemsetAsync(ctx->scal, 0, (4 + 2 * kPrepMaxBlocks) * sizeof(double), ctx->stream) != cudaSuccess) { rc = BANG_ECUDA; break; }
        if (cudaMalloc(&ctx->W_dev, ctx->W.size() * sizeof(double)) != cudaSuccess) { rc = BANG_ENOMEM; break; }
        if (cudaMemcpyAsync(ctx->W_dev, ctx->W.data(), ctx->W.size() * sizeof(double), cudaMemcpyHostToDevice, ctx->stream) != cudaSuccess ||
            cudaStreamSynchronize(ctx->stream) != cudaSuccess) { rc = BANG_ECUDA; break; }
        rc = f64 ? setup_slow<double>(ctx) : setup_slow<float>(ctx);
        if (rc != BANG_OK) break;
        // the allocation-free entry point's scratch: its device address on THIS device (current here: DeviceGuard above)
        if (noalloc_scratch_address(device, &ctx->na_scratch) != cudaSuccess) { rc = BANG_ECUDA; break; }
        // does the fused kernel fit (shared memory, registers)?
        FusedLaunch L = make_launch(ctx, nullptr, 1, 0, nullptr, nullptr);
        FusedInfo info{};
        cudaError_t e = dispatch_fused(ctx, L, &info, true);
        if (e != cudaSuccess) { rc = (e == cudaErrorInvalidValue || e == cudaErrorLaunchOutOfResources) ? BANG_EINVAL : BANG_ECUDA; break; }
    } while (0);
    if (rc != BANG_OK) { cudaGetLastError(); bang_destroy(ctx); return rc; }
    *out = ctx;
    return BANG_OK;
}

int bang_set_data(bang_ctx* ctx, const double* data_dev, const double* err_dev, const unsigned char* mask_dev) {
    if (!ctx) return BANG_EINVAL;
    if (!data_dev || !err_dev || !mask_dev) return fail(ctx, BANG_EINVAL, "bang_set_data: null pointer");
    ON_DEVICE(ctx);
    double2* buf = nullptr;
    const int gmax = data_gmax(ctx);
    const size_t n = (size_t)ctx->g.ny * 4 * ctx->P * gmax;
    CU(cudaMalloc(&buf, n * sizeof(double2)));
    CU(cudaMemsetAsync(buf, 0, n * sizeof(double2), ctx->stream));
    const int prep_total = ctx->g.ny * 4 * ctx->nxp;
    const int prep_blocks = std::max(1, std::min(kPrepMaxBlocks, (prep_total + 1023) / 1024));
    k_prep_data<<<prep_blocks, 256, 0, ctx->stream>>>(ctx->g.nx, ctx->g.ny, ctx->nxp, ctx->P, gmax, data_dev, err_dev, mask_dev, buf, ctx->scal,
                                                    reinterpret_cast<unsigned*>(ctx->scal + 2 + 2 * kPrepMaxBlocks));
    ctx->launches += 1;
    double scal[2] = {0, 0};
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaMemcpyAsync(scal, ctx->scal, sizeof(scal), cudaMemcpyDeviceToHost, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    if (e != cudaSuccess) { cudaFree(buf); return fail(ctx, BANG_ECUDA, "bang_set_data: %s", cudaGetErrorString(e)); }
    if (scal[1] != 0.0) {
        cudaFree(buf);
        return fail(ctx, BANG_EINVAL, "bang_set_data: %d used pixel(s) with err <= 0 or non-finite data/err", (int)scal[1]);
    }
    cudaFree(ctx->data);
    ctx->data = buf; ctx->C0 = scal[0]; ctx->has_data = true;
    return BANG_OK;
}

int bang_model_maps(bang_ctx* ctx, const double* theta_dev, int B, void* maps_dev) {
    if (!ctx) return BANG_EINVAL;
    if (B < 0 || (B > 0 && (!theta_dev || !maps_dev))) return fail(ctx, BANG_EINVAL, "bang_model_maps: bad arguments");
    if (B == 0) return BANG_OK;
    ON_DEVICE(ctx);
    int rc = ensure_slow_list(ctx, B);
    if (rc != BANG_OK) return rc;
    FusedLaunch L = make_launch(ctx, theta_dev, B, 0, maps_dev, nullptr);
    CU(dispatch_fused(ctx, L, nullptr, false));
    ctx->launches += 1;
    return ctx->model.precision == BANG_FP64 ? run_slow<double>(ctx, theta_dev, 0, maps_dev, nullptr)
                                             : run_slow<float>(ctx, theta_dev, 0, maps_dev, nullptr);
}

int bang_loglike(bang_ctx* ctx, const double* theta_dev, int B, double* logL_dev) {
    if (!ctx) return BANG_EINVAL;
    if (B < 0 || (B > 0 && (!theta_dev || !logL_dev))) return fail(ctx, BANG_EINVAL, "bang_loglike: bad arguments");
    if (!ctx->has_data) return fail(ctx, BANG_ENODATA, "bang_loglike: no data loaded");
    if (B == 0) return BANG_OK;
    ON_DEVICE(ctx);
    int rc = ensure_slow_list(ctx, B);
    if (rc != BANG_OK) return rc;
    FusedLaunch L = make_launch(ctx, theta_dev, B, 1, nullptr, logL_dev);
    CU(dispatch_fused(ctx, L, nullptr, false));
    ctx->launches += 1;
    return ctx->model.precision == BANG_FP64 ? run_slow<double>(ctx, theta_dev, 1, nullptr, logL_dev)
                                             : run_slow<float>(ctx, theta_dev, 1, nullptr, logL_dev);
}

int bang_loglike_noalloc(bang_ctx* ctx, const double* theta_dev, int B, double* logL_dev) {
    if (!ctx) return BANG_EINVAL;
    if (B < 0 || (B > 0 && (!theta_dev || !logL_dev))) return fail(ctx, BANG_EINVAL, "bang_loglike_noalloc: bad arguments");
    if (B > BANG_NOALLOC_MAX_B)
        return fail(ctx, BANG_EINVAL, "bang_loglike_noalloc: B = %d exceeds BANG_NOALLOC_MAX_B = %d (the static scratch holds one "
                                      "list entry per theta); split the batch or call bang_loglike", B, BANG_NOALLOC_MAX_B);
    if (!ctx->has_data) return fail(ctx, BANG_ENODATA, "bang_loglike_noalloc: no data loaded");
    if (!ctx->na_scratch) return fail(ctx, BANG_ECUDA, "bang_loglike_noalloc: the scratch symbol has no address on device %d", ctx->device);
    if (B == 0) return BANG_OK;
    ON_DEVICE(ctx);
    // the array keeps the last call's contents: the two counters must start at zero (k_slow resets them when it finishes,
    // but a call that failed half-way, or another context's, may not have)
    CU(cudaMemsetAsync(ctx->na_scratch, 0, 64 * sizeof(int), ctx->stream));
    FusedLaunch L = make_launch(ctx, theta_dev, B, 1, nullptr, logL_dev);
    L.slow_list = ctx->slow_smem ? ctx->na_scratch + 64 : nullptr;
    L.slow_count = ctx->na_scratch;
    CU(dispatch_fused(ctx, L, nullptr, false));
    ctx->launches += 1;
    return ctx->model.precision == BANG_FP64 ? run_slow_noalloc<double>(ctx, theta_dev, logL_dev)
                                             : run_slow_noalloc<float>(ctx, theta_dev, logL_dev);
}

int bang_ns_walk(bang_ctx* ctx, int K, int d, const int* free_idx_host, const double* lo_host, const double* hi_host,
                 const double* theta0_host, double* u_dev, double* logL_dev, const double* Lstar_dev, const int* group_dev,
                 int n_groups, const double* chol_host, const double* scale_host, int steps, unsigned long long seed,
                 int* n_accept_host) {
    if (!ctx) return BANG_EINVAL;
    if (K < 0 || d < 1 || d > kNsMaxDim || n_groups < 1 || steps < 0 || !free_idx_host || !lo_host || !hi_host || !theta0_host ||
        !chol_host || !scale_host || !n_accept_host || (K > 0 && (!u_dev || !logL_dev || !Lstar_dev || !group_dev)))
        return fail(ctx, BANG_EINVAL, "bang_ns_walk: bad arguments");
    for (int j = 0; j < d; ++j)
        if (free_idx_host[j] < 0 || free_idx_host[j] >= kNTheta) return fail(ctx, BANG_EINVAL, "bang_ns_walk: free index out of range");
    if (!ctx->has_data) return fail(ctx, BANG_ENODATA, "bang_ns_walk: no data loaded");
    for (int g = 0; g < n_groups; ++g) n_accept_host[g] = 0;
    if (K == 0 || steps == 0) return BANG_OK;
    ON_DEVICE(ctx);
    if (K > ctx->ns_capK) {
        CU(cudaStreamSynchronize(ctx->stream));
        cudaFree(ctx->ns_prop); cudaFree(ctx->ns_theta); cudaFree(ctx->ns_pl);
        ctx->ns_prop = ctx->ns_theta = ctx->ns_pl = nullptr; ctx->ns_capK = 0;
        CU(cudaMalloc(&ctx->ns_prop, (size_t)K * kNsMaxDim * sizeof(double)));
        CU(cudaMalloc(&ctx->ns_theta, (size_t)K * kNTheta * sizeof(double)));
        CU(cudaMalloc(&ctx->ns_pl, (size_t)K * sizeof(double)));
        ctx->ns_capK = K;
    }
    if (n_groups > ctx->ns_capG) {
        CU(cudaStreamSynchronize(ctx->stream));
        cudaFree(ctx->ns_chol); cudaFree(ctx->ns_acc);
        ctx->ns_chol = nullptr; ctx->ns_acc = nullptr; ctx->ns_capG = 0;
        CU(cudaMalloc(&ctx->ns_chol, (size_t)n_groups * (kNsMaxDim * kNsMaxDim + 1) * sizeof(double)));
        CU(cudaMalloc(&ctx->ns_acc, (size_t)n_groups * sizeof(int)));
        ctx->ns_capG = n_groups;
    }
    // Cholesky factors then scales (times the random-walk Metropolis factor 2.38/sqrt(d)), one small synchronous copy
    std::vector<double> cs((size_t)n_groups * d * d + n_groups);
    memcpy(cs.data(), chol_host, (size_t)n_groups * d * d * sizeof(double));
    for (int g = 0; g < n_groups; ++g) cs[(size_t)n_groups * d * d + g] = scale_host[g] * 2.38 / std::sqrt((double)d);
    CU(cudaMemcpyAsync(ctx->ns_chol, cs.data(), cs.size() * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));                          // cs is pageable host memory: done before it goes away
    CU(cudaMemsetAsync(ctx->ns_acc, 0, (size_t)n_groups * sizeof(int), ctx->stream));
    NsParams p{};
    p.K = K; p.d = d; p.seed = seed;
    for (int j = 0; j < d; ++j) { p.free_idx[j] = free_idx_host[j]; p.lo[j] = lo_host[j]; p.hi[j] = hi_host[j]; }
    for (int i = 0; i < kNTheta; ++i) p.theta0[i] = theta0_host[i];
    p.u = u_dev; p.logL = logL_dev; p.Lstar = Lstar_dev; p.group = group_dev;
    p.chol = ctx->ns_chol; p.scale = ctx->ns_chol + (size_t)n_groups * d * d;
    p.prop = ctx->ns_prop; p.theta = ctx->ns_theta;
    const int th = 128, blocks = (K + th - 1) / th;
    for (int step = 0; step < steps; ++step) {
        p.step = step;
        k_ns_propose<<<blocks, th, 0, ctx->stream>>>(p);
        int rc = bang_loglike(ctx, ctx->ns_theta, K, ctx->ns_pl);
        if (rc != BANG_OK) return rc;
        k_ns_accept<<<blocks, th, 0, ctx->stream>>>(K, d, ctx->ns_prop, ctx->ns_pl, Lstar_dev, group_dev, u_dev, logL_dev, ctx->ns_acc);
        ctx->launches += 2;
    }
    CU(cudaGetLastError());
    CU(cudaMemcpyAsync(n_accept_host, ctx->ns_acc, (size_t)n_groups * sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    return BANG_OK;
}

int bang_model_fine(bang_ctx* ctx, const double* theta_dev, int B, void* fine_dev) {
    if (!ctx) return BANG_EINVAL;
    if (B < 0 || (B > 0 && (!theta_dev || !fine_dev))) return fail(ctx, BANG_EINVAL, "bang_model_fine: bad arguments");
    if (B == 0) return BANG_OK;
    ON_DEVICE(ctx);
    const bool f64 = ctx->model.precision == BANG_FP64;
    const int ctas = std::min(B, 8 * ctx->n_sm);
    const DirectC direct = make_direct(ctx);
    if (f64) {
        FineParams<double> p{ctx->g, ctx->fit,
                             PolyTab<double>{static_cast<const double*>(ctx->btab), ctx->btab_first, ctx->btab_cells},
                             PolyTab<double>{static_cast<const double*>(ctx->Ftab), ctx->Ftab_first, ctx->Ftab_cells},
                             direct, (int)bs_elems<double>(ctx->g), theta_dev, B, static_cast<double*>(fine_dev)};
        const size_t smem = fused_smem_bytes<double>(ctx->g, 0, 0);
        if (!ctx->fine_ready) CU(cudaFuncSetAttribute(k_fine<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, ctx->smem_optin));
        k_fine<double><<<ctas, 256, smem, ctx->stream>>>(p);
    } else {
        FineParams<float> p{ctx->g, ctx->fit,
                            PolyTab<float>{static_cast<const float*>(ctx->btab), ctx->btab_first, ctx->btab_cells},
                            PolyTab<float>{static_cast<const float*>(ctx->Ftab), ctx->Ftab_first, ctx->Ftab_cells},
                            direct, (int)bs_elems<float>(ctx->g), theta_dev, B, static_cast<float*>(fine_dev)};
        const size_t smem = fused_smem_bytes<float>(ctx->g, 0, 0);
        if (!ctx->fine_ready) CU(cudaFuncSetAttribute(k_fine<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, ctx->smem_optin));
        k_fine<float><<<ctas, 256, smem, ctx->stream>>>(p);
    }
    ctx->launches += 1;
    CU(cudaGetLastError());
    ctx->fine_ready = true;
    return BANG_OK;
}

int bang_loglike_host(bang_ctx* ctx, const double* theta_host, int B, double* logL_host) {
    if (!ctx) return BANG_EINVAL;
    if (B < 0 || (B > 0 && (!theta_host || !logL_host))) return fail(ctx, BANG_EINVAL, "bang_loglike_host: bad arguments");
    if (!ctx->has_data) return fail(ctx, BANG_ENODATA, "bang_loglike_host: no data loaded");
    if (B == 0) return BANG_OK;
    ON_DEVICE(ctx);
    int rc = ensure_staging(ctx, B, (size_t)B * sizeof(double));
    if (rc != BANG_OK) return rc;
    const size_t tb = (size_t)B * kNTheta * sizeof(double);
    memcpy(ctx->h_theta, theta_host, tb);
    CU(cudaMemcpyAsync(ctx->d_theta, ctx->h_theta, tb, cudaMemcpyHostToDevice, ctx->stream));
    rc = bang_loglike(ctx, ctx->d_theta, B, static_cast<double*>(ctx->d_out));
    if (rc != BANG_OK) return rc;
    CU(cudaMemcpyAsync(ctx->h_out, ctx->d_out, (size_t)B * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    memcpy(logL_host, ctx->h_out, (size_t)B * sizeof(double));
    return BANG_OK;
}

int bang_model_maps_host(bang_ctx* ctx, const double* theta_host, int B, void* maps_host) {
    if (!ctx) return BANG_EINVAL;
    if (B < 0 || (B > 0 && (!theta_host || !maps_host))) return fail(ctx, BANG_EINVAL, "bang_model_maps_host: bad arguments");
    if (B == 0) return BANG_OK;
    ON_DEVICE(ctx);
    const size_t esz = ctx->model.precision == BANG_FP64 ? 8 : 4;
    const size_t ob = (size_t)B * 4 * ctx->g.nx * ctx->g.ny * esz;
    int rc = ensure_staging(ctx, B, ob);
    if (rc != BANG_OK) return rc;
    const size_t tb = (size_t)B * kNTheta * sizeof(double);
    memcpy(ctx->h_theta, theta_host, tb);
    CU(cudaMemcpyAsync(ctx->d_theta, ctx->h_theta, tb, cudaMemcpyHostToDevice, ctx->stream));
    rc = bang_model_maps(ctx, ctx->d_theta, B, ctx->d_out);
    if (rc != BANG_OK) return rc;
    CU(cudaMemcpyAsync(ctx->h_out, ctx->d_out, ob, cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    memcpy(maps_host, ctx->h_out, ob);
    return BANG_OK;
}

}  // extern "C"
