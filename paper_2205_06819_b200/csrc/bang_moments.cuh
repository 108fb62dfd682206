// bang_moments.cuh -- the flux-weighted PSF variant (reading G'; BANG_PSF_FLUX), run unfused.  Included by bang_api.cu only.
#pragma once
#include "bang_kernels.cuh"

namespace bang {

// ---- flux-weighted PSF variant (reading G'; BANG_PSF_FLUX), UNFUSED: k_fine writes the four moment fields of a chunk of
// theta to HBM, this kernel applies the composite taps (box_s (*) Gaussian at stride s, W[0 .. 2 r_k + s)) along x and y,
// forms B = M0, v = M1/M0, sigma^2 = M2/M0 - v^2, M/L = M3/M0 per data pixel and stores the maps or reduces eq. 18.
// One CTA per (theta, data row); thread = data column.  A side variant: HBM-bound (16 B per fine cell each way), kept out
// of the fused kernel so that the paper's path carries none of its code.
template <typename T>
struct MomentsParams {
    GridC g;
    int ntap;                    // 2 r_k + s
    const double* W;             // [ntap] composite taps (device)
    const T* fine;               // [Bc][4][nfy][nfx] moment fields
    int Bc, b0;                  // chunk size, index of its first theta in the batch
    const int* valid;            // [Bc] 0 = out-of-domain theta
    T* maps;                     // [B][4][ny][nx]   (mode 0)
    const double2* data;         // [ny][4][P][gmax] {d, 1/e}
    int P, gmax;
    double* chi2;                // [B][ny] partial chi-squares (mode 1), reduced by k_moments_reduce
    int mode;
};
template <typename T>
__global__ void __launch_bounds__(256) k_psf_moments(const __grid_constant__ MomentsParams<T> p) {
    __shared__ double red[8];
    const GridC& g = p.g;
    const int bl = blockIdx.x / g.ny, py = blockIdx.x - bl * g.ny, b = p.b0 + bl;
    const size_t plane = (size_t)g.nfx * g.nfy, npix = (size_t)g.nx * g.ny;
    double z2 = 0.0;
    for (int px = threadIdx.x; px < g.nx; px += blockDim.x) {
        T out[4];
        if (!p.valid[bl]) {
            out[0] = out[1] = out[2] = out[3] = (T)nan("");
        } else {
            double M[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const T* f = p.fine + ((size_t)bl * 4 + q) * plane + (size_t)(py * g.s) * g.nfx + px * g.s;
                double a = 0.0;
                for (int ty = 0; ty < p.ntap; ++ty) {
                    double r = 0.0;
                    for (int tx = 0; tx < p.ntap; ++tx) r = fma(p.W[tx], (double)f[(size_t)ty * g.nfx + tx], r);
                    a = fma(p.W[ty], r, a);
                }
                M[q] = a;
            }
            const double i0 = 1.0 / fmax(M[0], 1e-300), v = M[1] * i0;
            out[0] = (T)M[0]; out[1] = (T)v; out[2] = (T)sqrt(fmax(M[2] * i0 - v * v, 0.0)); out[3] = (T)(M[3] * i0);
        }
        if (p.mode == 0) {
#pragma unroll
            for (int q = 0; q < 4; ++q) p.maps[((size_t)b * 4 + q) * npix + (size_t)py * g.nx + px] = out[q];
        } else {
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const double2 de = p.data[(((size_t)py * 4 + q) * p.P + px % p.P) * p.gmax + px / p.P];
                const double z = (de.x - (double)out[q]) * de.y;
                z2 = (de.y != 0.0) ? fma(z, z, z2) : z2;
            }
        }
    }
    if (p.mode == 1) {                               // fixed-order block reduction
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) z2 += __shfl_xor_sync(0xffffffffu, z2, o);
        if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = z2;
        __syncthreads();
        if (threadIdx.x == 0) {
            double sum = 0.0;
            for (int w = 0; w < (int)(blockDim.x + 31) / 32; ++w) sum += red[w];
            p.chi2[(size_t)b * g.ny + py] = sum;
        }
    }
}
// logL[b] = C0 - 1/2 sum over rows of the partial chi-squares (or -inf for an out-of-domain theta); fixed order
__global__ void k_moments_reduce(const double* __restrict__ chi2, const int* __restrict__ valid, int Bc, int b0, int ny,
                                 double C0, double* __restrict__ logL) {
    const int bl = blockIdx.x * blockDim.x + threadIdx.x;
    if (bl >= Bc) return;
    double sum = 0.0;
    for (int r = 0; r < ny; ++r) sum += chi2[(size_t)(b0 + bl) * ny + r];
    logL[b0 + bl] = valid[bl] ? C0 - 0.5 * sum : -INFINITY;
}
// validity of each theta of a chunk (the decode's verdict), for the kernels above
template <typename T>
__global__ void k_theta_valid(const double* __restrict__ theta, int Bc, GridC g, PolyTab<T> btab, PolyTab<T> Ftab, int* __restrict__ valid) {
    const int bl = blockIdx.x * blockDim.x + threadIdx.x;
    if (bl >= Bc) return;
    ThetaC<T> c;
    decode_theta<T>(theta + (size_t)bl * kNTheta, g, btab, Ftab, c);
    valid[bl] = c.valid;
}

}  // namespace bang
